// Fused ramp filter (include/pyhst.h a1; NEXT row N2 of SURVEY.md sec. 8(f): "fused smem FFT filter:
// pad, FFT, x H, IFFT, crop in one kernel at the 8 B/sample HBM floor"; readings R8, R9).
//
// One thread block filters FOUR real rows -- the four slices of one slice group at one projection when
// it writes the backprojector's interleaved layout, four consecutive rows otherwise -- as TWO complex
// sequences z = a + i b of length M = 2^L >= 2 n_bins_out held in shared memory: the ramp kernel h is
// real, so conv(a + i b, h) = conv(a, h) + i conv(b, h) and nothing has to be unpacked.  Per block:
//   raw rows (x column weights) -> shared memory at offset pad_left, zeros elsewhere
//   forward FFT: in-place decimation in frequency, radix 8 (last pass radix 4 or 2), natural order in,
//                digit-reversed order out
//   x H: fused into the last forward pass; the table Hq[pos] = H[frequency at position pos] / M is made
//        once per (filter, M) on the host in double (closed-form h, double FFT) -- no reordering pass
//   inverse FFT: the same passes backwards with conjugate twiddles (decimation in time), natural order out
//   crop: bins [0, n_bins_out) written once, as plain rows or as float4 of the interleaved layout
// HBM traffic = one read of the raw rows + one write of the filtered rows (the cuFFT path makes five
// passes over a padded buffer).  Twiddles exp(-2 pi i k / M) come from a table computed in double.
// The cuFFT path (filter.cu) stays selectable (pyhst_test.h: pyhst_set_filter_variant) as a cross-check.
#include <cmath>
#include <complex>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

#include "common.h"

namespace pyhst {

namespace {

#ifndef FF_SQUARE_TW
#define FF_SQUARE_TW 1
#endif
constexpr int FF_MAX_LOG2 = 13;   // M <= 8192: 2 sequences x 9/8 M x 8 B = 144 KB of shared memory

__device__ __forceinline__ int ff_phys(int i) { return i + (i >> 3); }   // one pad per 8 complex: no bank conflicts
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiply by -i (forward) or +i (inverse)
template <bool INV>
__device__ __forceinline__ float2 crot(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

// R-point DFT in registers, forward (e^{-2 pi i / R}) or inverse (conjugate), output index = frequency
template <int R, bool INV>
__device__ __forceinline__ void small_dft(float2 (&v)[R]) {
  if (R == 2) {
    const float2 a = cadd(v[0], v[1]), b = csub(v[0], v[1]);
    v[0] = a;
    v[1] = b;
  } else if (R == 4) {
    const float2 d0 = cadd(v[0], v[2]), d1 = cadd(v[1], v[3]), d2 = csub(v[0], v[2]),
                 d3 = crot<INV>(csub(v[1], v[3]));
    v[0] = cadd(d0, d1);
    v[2] = csub(d0, d1);
    v[1] = cadd(d2, d3);
    v[3] = csub(d2, d3);
  } else {
    const float h = 0.70710678118654752f;
    const float2 a0 = cadd(v[0], v[4]), a4 = csub(v[0], v[4]);
    const float2 a1 = cadd(v[1], v[5]);
    float2 a5 = csub(v[1], v[5]);
    const float2 a2 = cadd(v[2], v[6]), a6 = crot<INV>(csub(v[2], v[6]));
    const float2 a3 = cadd(v[3], v[7]);
    float2 a7 = csub(v[3], v[7]);
    // a5 *= w8, a7 *= w8^3 (w8 = e^{-+ i pi / 4})
    a5 = INV ? make_float2(h * (a5.x - a5.y), h * (a5.x + a5.y)) : make_float2(h * (a5.x + a5.y), h * (a5.y - a5.x));
    a7 = INV ? make_float2(-h * (a7.x + a7.y), h * (a7.x - a7.y)) : make_float2(h * (a7.y - a7.x), -h * (a7.x + a7.y));
    const float2 b0 = cadd(a0, a2), b2 = csub(a0, a2), b1 = cadd(a1, a3), b3 = crot<INV>(csub(a1, a3));
    const float2 b4 = cadd(a4, a6), b6 = csub(a4, a6), b5 = cadd(a5, a7), b7 = crot<INV>(csub(a5, a7));
    v[0] = cadd(b0, b1);
    v[4] = csub(b0, b1);
    v[2] = cadd(b2, b3);
    v[6] = csub(b2, b3);
    v[1] = cadd(b4, b5);
    v[5] = csub(b4, b5);
    v[3] = cadd(b6, b7);
    v[7] = csub(b6, b7);
  }
}

// powers w^1 .. w^{R-1} of w = tw[k]: one table read, w^2 and w^4 by squaring (two roundings more on those two
// factors, ~2e-7 relative: the filter stays at rel-L2 3e-7 against the oracle) -- the three dependent global reads
// per butterfly were the kernel's top stall (long_scoreboard); FF_SQUARE_TW = 0 restores the table reads
template <int R>
__device__ __forceinline__ void twiddle_powers(const float2* __restrict__ tw, int k, float2 (&w)[R]) {
  w[0] = make_float2(1.f, 0.f);
  w[1] = tw[k];
  if (R >= 4) {
    w[2] = FF_SQUARE_TW ? cmul(w[1], w[1]) : tw[2 * k];
    w[3] = cmul(w[1], w[2]);
  }
  if (R == 8) {
    w[4] = FF_SQUARE_TW ? cmul(w[2], w[2]) : tw[4 * k];
    w[5] = cmul(w[1], w[4]);
    w[6] = cmul(w[2], w[4]);
    w[7] = cmul(w[3], w[4]);
  }
}

// One pass over both sequences.  Sub-transform size n, radix R, s = n / R: butterfly (blk, j) works on the
// elements blk n + j + q s.  Forward: DFT across q, then output r times w_n^{r j} (and Hq when given).
// Inverse: input r times conj(w_n^{r j}), then the inverse DFT.
template <int R, bool INV>
__device__ __forceinline__ void ff_pass(float2* sm, int seq_stride, int M, int log2n, const float2* __restrict__ tw,
                                        const float* __restrict__ Hq) {
  const int log2s = log2n - (R == 8 ? 3 : (R == 4 ? 2 : 1));
  const int s = 1 << log2s, per_seq = M / R;
  const int tstride = M >> log2n;   // table index of w_n
  for (int t = threadIdx.x; t < 2 * per_seq; t += blockDim.x) {
    const int seq = t >= per_seq ? 1 : 0;
    const int tt = t - seq * per_seq;
    const int blk = tt >> log2s, j = tt & (s - 1);
    const int base = (blk << log2n) + j;
    float2* x = sm + seq * seq_stride;
    float2 v[R], w[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = x[ff_phys(base + q * s)];
    twiddle_powers<R>(tw, j * tstride, w);
    if (INV) {
#pragma unroll
      for (int r = 1; r < R; ++r) v[r] = cmul(v[r], cconj(w[r]));
      small_dft<R, true>(v);
    } else {
      small_dft<R, false>(v);
#pragma unroll
      for (int r = 1; r < R; ++r) v[r] = cmul(v[r], w[r]);
      if (Hq) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const float hh = Hq[base + r * s];
          v[r].x *= hh;
          v[r].y *= hh;
        }
      }
    }
#pragma unroll
    for (int q = 0; q < R; ++q) x[ff_phys(base + q * s)] = v[q];
  }
  __syncthreads();
}

struct FusedArgs {
  const float* in;            // rows [.. ][in_pitch]
  int64_t in_pitch;
  const float* w;             // column weights or NULL
  int n_bins_in, n_bins_out, pad_left, log2M;
  const float2* tw;           // [M]
  const float* Hq;            // [M], H at the position's frequency, / M
  // plain rows
  float* out;
  int64_t out_pitch, n_rows;
  // interleaved layout of one slice group (d_qi already offset to the group)
  float4* qi;
  int64_t row_f4;
  int zpad, n_angles, n_slices_in;   // n_slices_in: slices of the whole stack; group blockIdx.y holds 4 of them
  int64_t in_group_floats, qi_group_f4;
  const uint8_t* flip;
};

__global__ void __launch_bounds__(1024) ramp_fused_kernel(FusedArgs a) {
  extern __shared__ float2 sm[];
  const int M = 1 << a.log2M;
  const int seq_stride = M + (M >> 3);
  const bool to_qi = a.qi != nullptr;
  if (to_qi) {   // blockIdx.y = slice group
    a.in += (int64_t)blockIdx.y * a.in_group_floats;
    a.qi += (int64_t)blockIdx.y * a.qi_group_f4;
    a.n_slices_in = min(4, a.n_slices_in - 4 * (int)blockIdx.y);
  }
  // the block's four rows
  int64_t row[4];
  bool have[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (to_qi) {
      row[k] = (int64_t)k * a.n_angles + blockIdx.x;
      have[k] = k < a.n_slices_in;
    } else {
      row[k] = (int64_t)blockIdx.x * 4 + k;
      have[k] = row[k] < a.n_rows;
    }
  }
  // ---- load: z[seq][pad_left + m] = (row 2 seq, row 2 seq + 1), zero elsewhere
  for (int i = threadIdx.x; i < M; i += blockDim.x) {
    const int m = i - a.pad_left;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (m >= 0 && m < a.n_bins_in) {
      const float cw = a.w ? a.w[m] : 1.f;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (have[k]) v[k] = a.in[row[k] * a.in_pitch + m] * cw;
    }
    sm[ff_phys(i)] = make_float2(v[0], v[1]);
    sm[seq_stride + ff_phys(i)] = make_float2(v[2], v[3]);
  }
  __syncthreads();
  // ---- forward (DIF), x Hq in the last pass
  const int n8 = a.log2M / 3, rem = a.log2M - 3 * n8;
  int log2n = a.log2M;
  for (int st = 0; st < n8; ++st) {
    ff_pass<8, false>(sm, seq_stride, M, log2n, a.tw, (rem == 0 && st == n8 - 1) ? a.Hq : nullptr);
    log2n -= 3;
  }
  if (rem == 2) ff_pass<4, false>(sm, seq_stride, M, log2n, a.tw, a.Hq);
  if (rem == 1) ff_pass<2, false>(sm, seq_stride, M, log2n, a.tw, a.Hq);
  // ---- inverse (DIT): the same passes backwards
  if (rem == 2) ff_pass<4, true>(sm, seq_stride, M, 2, a.tw, nullptr);
  if (rem == 1) ff_pass<2, true>(sm, seq_stride, M, 1, a.tw, nullptr);
  log2n = rem + 3;
  for (int st = 0; st < n8; ++st) {
    ff_pass<8, true>(sm, seq_stride, M, log2n, a.tw, nullptr);
    log2n += 3;
  }
  // ---- crop / interleave
  if (to_qi) {
    const int p = blockIdx.x;
    const bool fl = a.flip && a.flip[p];
    float4* dst = a.qi + (int64_t)p * a.row_f4;
    for (int64_t x = threadIdx.x; x < a.row_f4; x += blockDim.x) {
      int64_t b = x - a.zpad;
      float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
      if (b >= 0 && b < a.n_bins_out) {
        if (fl) b = a.n_bins_out - 1 - b;      // reversed row, see bp_run_kernel
        const float2 u = sm[ff_phys((int)b)], v = sm[seq_stride + ff_phys((int)b)];
        o = make_float4(u.x, u.y, v.x, v.y);
      }
      dst[x] = o;
    }
  } else {
    for (int b = threadIdx.x; b < a.n_bins_out; b += blockDim.x) {
      const float2 u = sm[ff_phys(b)], v = sm[seq_stride + ff_phys(b)];
      if (have[0]) a.out[row[0] * a.out_pitch + b] = u.x;
      if (have[1]) a.out[row[1] * a.out_pitch + b] = u.y;
      if (have[2]) a.out[row[2] * a.out_pitch + b] = v.x;
      if (have[3]) a.out[row[3] * a.out_pitch + b] = v.y;
    }
  }
}

// ---- host: tables per (device, filter, log2M) ---------------------------------------------------
void host_fft(std::vector<std::complex<double>>& x) {   // in-place radix-2, natural order in and out
  const size_t n = x.size();
  for (size_t i = 1, j = 0; i < n; ++i) {
    size_t bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(x[i], x[j]);
  }
  const double PI = 3.14159265358979323846264338327950288;
  for (size_t len = 2; len <= n; len <<= 1) {
    for (size_t i = 0; i < n; i += len)
      for (size_t k = 0; k < len / 2; ++k) {
        const double ang = -2.0 * PI * (double)k / (double)len;
        const std::complex<double> w(std::cos(ang), std::sin(ang));
        const std::complex<double> u = x[i + k], v = x[i + k + len / 2] * w;
        x[i + k] = u + v;
        x[i + k + len / 2] = u - v;
      }
  }
}

double ramp_tap(int filter, int64_t l) {   // h[l] of R8 / R8c in double (same closed forms as filter.cu)
  const double PI = 3.14159265358979323846264338327950288;
  auto ramlak = [PI](int64_t m) {
    const double dm = (double)m;
    return m == 0 ? 0.25 : ((m & 1) ? -1.0 / (PI * PI * dm * dm) : 0.0);
  };
  const double dl = (double)l;
  if (filter == PYHST_FILTER_RAMLAK) return ramlak(l);
  if (filter == PYHST_FILTER_SHEPP_LOGAN) return -2.0 / (PI * PI * (4.0 * dl * dl - 1.0));
  if (filter == PYHST_FILTER_COSINE) {
    auto half_shifted = [PI](int64_t m) {
      const double x = (double)m + 0.5;
      return ((m & 1) ? -1.0 : 1.0) / (2.0 * PI * x) - 1.0 / (2.0 * PI * PI * x * x);
    };
    return 0.5 * (half_shifted(l - 1) + half_shifted(l));
  }
  const double a0 = filter == PYHST_FILTER_HANN ? 0.5 : 0.54, a1 = filter == PYHST_FILTER_HANN ? 0.25 : 0.23;
  return a0 * ramlak(l) + a1 * (ramlak(l - 1) + ramlak(l + 1));
}

struct FusedTables { float2* d_tw = nullptr; float* d_Hq = nullptr; };
std::mutex g_mu;
std::map<std::tuple<int, int, int>, FusedTables> g_tables;   // (device, filter, log2M)
std::map<std::pair<int, int>, float2*> g_twiddles;           // (device, log2M)

int get_tables(int filter, int log2M, cudaStream_t stream, FusedTables* out) {
  std::lock_guard<std::mutex> lock(g_mu);
  const int dev = current_device();
  auto key = std::make_tuple(dev, filter, log2M);
  auto it = g_tables.find(key);
  if (it != g_tables.end()) { *out = it->second; return PYHST_OK; }
  const int M = 1 << log2M;
  const double PI = 3.14159265358979323846264338327950288;
  FusedTables t;
  auto tk = std::make_pair(dev, log2M);
  auto itw = g_twiddles.find(tk);
  if (itw != g_twiddles.end()) {
    t.d_tw = itw->second;
  } else {
    std::vector<float2> tw((size_t)M);
    for (int k = 0; k < M; ++k) {
      const double ang = -2.0 * PI * (double)k / (double)M;
      tw[k] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
    PYHST_CUDA_TRY(cudaMalloc(&t.d_tw, sizeof(float2) * M));
    PYHST_CUDA_TRY(cudaMemcpyAsync(t.d_tw, tw.data(), sizeof(float2) * M, cudaMemcpyHostToDevice, stream));
    PYHST_CUDA_TRY(cudaStreamSynchronize(stream));   // pageable source; one-time set-up
    g_twiddles[tk] = t.d_tw;
  }
  // H = DFT_M(hc), hc[l mod M] = h[l] for -M/2 < l <= M/2 (R8, R9): real and even
  std::vector<std::complex<double>> hc((size_t)M);
  for (int n = 0; n < M; ++n) hc[n] = ramp_tap(filter, n <= M / 2 ? n : n - M);
  host_fft(hc);
  // frequency held at position pos after the forward passes: the digits of pos, most significant first
  // (one per pass), are the output indices r of the passes; frequency = sum r_i * (product of the earlier radices)
  std::vector<float> Hq((size_t)M);
  const int n8 = log2M / 3, rem = log2M - 3 * n8;
  for (int pos = 0; pos < M; ++pos) {
    int left = pos, n = M, freq = 0, mult = 1;
    for (int st = 0; st < n8 + (rem ? 1 : 0); ++st) {
      const int R = st < n8 ? 8 : (rem == 2 ? 4 : 2);
      const int s = n / R, r = left / s;
      left -= r * s;
      freq += r * mult;
      mult *= R;
      n = s;
    }
    Hq[pos] = (float)(hc[(size_t)freq].real() / (double)M);
  }
  PYHST_CUDA_TRY(cudaMalloc(&t.d_Hq, sizeof(float) * M));
  PYHST_CUDA_TRY(cudaMemcpyAsync(t.d_Hq, Hq.data(), sizeof(float) * M, cudaMemcpyHostToDevice, stream));
  PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
  g_tables[key] = t;
  *out = t;
  return PYHST_OK;
}

}  // namespace

// log2 of the FFT length the fused kernel would use for rows of n_bins_out, 0 if it does not cover them
int ramp_fused_log2m(int32_t n_bins_out) {
  int l = 6;
  while ((1 << l) < 2 * (int64_t)n_bins_out && l <= FF_MAX_LOG2) ++l;
  return l <= FF_MAX_LOG2 ? l : 0;
}

int launch_ramp_filter_fused(const float* d_in, int64_t in_pitch, int64_t n_rows, int32_t n_bins_in,
                             int32_t n_bins_out, int32_t pad_left, int filter, const float* d_col_weights,
                             float* d_out, int64_t out_pitch, float4* d_qi, const QiLayout* L, int32_t n_slices_in,
                             const uint8_t* d_flip, cudaStream_t stream) {
  if (n_rows == 0) return PYHST_OK;
  const int log2M = ramp_fused_log2m(n_bins_out);
  if (!log2M) return set_error(PYHST_ERR_UNSUPPORTED, "fused ramp filter: rows of %d bins are too long", n_bins_out);
  FusedTables t;
  PYHST_TRY(get_tables(filter, log2M, stream, &t));
  const int M = 1 << log2M;
  const size_t smem = (size_t)2 * (M + (M >> 3)) * sizeof(float2);
  static PerDeviceSize configured;
  if (smem > configured.here()) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(ramp_fused_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured.here() = smem;
  }
  FusedArgs a{};
  a.in = d_in;
  a.in_pitch = in_pitch;
  a.w = d_col_weights;
  a.n_bins_in = n_bins_in;
  a.n_bins_out = n_bins_out;
  a.pad_left = pad_left;
  a.log2M = log2M;
  a.tw = t.d_tw;
  a.Hq = t.d_Hq;
  unsigned blocks, groups = 1;
  if (d_qi) {
    // n_slices_in slices = ceil(n_slices_in / 4) slice groups, all in one launch (rows of group g start
    // 4 g n_angles rows further on)
    a.qi = d_qi;
    a.row_f4 = L->row_f4();
    a.zpad = L->zpad;
    a.n_angles = L->n_angles;
    a.n_slices_in = n_slices_in;
    a.in_group_floats = (int64_t)4 * L->n_angles * in_pitch;
    a.qi_group_f4 = L->group_f4();
    a.flip = d_flip;
    blocks = (unsigned)L->n_angles;
    groups = (unsigned)((n_slices_in + 3) / 4);
  } else {
    a.out = d_out;
    a.out_pitch = out_pitch;
    a.n_rows = n_rows;
    if ((n_rows + 3) / 4 > 0x7fffffff) return set_error(PYHST_ERR_UNSUPPORTED, "fused ramp filter: too many rows");
    blocks = (unsigned)((n_rows + 3) / 4);
  }
  const int nt = M >= 8192 ? 1024 : (M >= 1024 ? 256 : 128);
  StageScope scope(ST_FILTER, stream);
  scope.kernels();
  ramp_fused_kernel<<<dim3(blocks, groups), nt, smem, stream>>>(a);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

void release_fused_filter_tables(int device) {
  std::lock_guard<std::mutex> lock(g_mu);
  for (auto it = g_tables.begin(); it != g_tables.end();) {
    if (std::get<0>(it->first) != device) { ++it; continue; }
    cudaFree(it->second.d_Hq);
    it = g_tables.erase(it);
  }
  for (auto it = g_twiddles.begin(); it != g_twiddles.end();) {
    if (it->first.first != device) { ++it; continue; }
    cudaFree(it->second);
    it = g_twiddles.erase(it);
  }
}

}  // namespace pyhst
