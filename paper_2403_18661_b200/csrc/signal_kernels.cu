// Welch periodograms, PSD mean, whitening-filter design and overlap-save whitening kernels.
//
//  O-1 (reading A1)  welch_periodogram_kernel + psd_mean_kernel
//  O-2 (readings A3-A6)            filter_design_kernel (double precision, one CTA per epoch x channel)
//  (O-3, the overlap-save whitening, lives in signal_fft64.cu)
#include "fft.cuh"
#include <atomic>

// --------------------------------------------------------------------------------------------------
// Welch: one CTA per (segment, channel).  NFFT real samples -> M = NFFT/2 complex FFT -> |X|^2.
// --------------------------------------------------------------------------------------------------
template <int NFFT>
__global__ void __launch_bounds__(NFFT / 32)
welch_periodogram_kernel(const float* __restrict__ strain, int64_t ld, int64_t hop, int64_t first_seg,
                         int64_t seg_stride_out, float scale, float norm, const float2* __restrict__ tw,
                         float* __restrict__ pgram, StreamGate gate) {
  constexpr int M = NFFT / 2;
  constexpr int NT = NFFT / 32;        // M / 16
  constexpr int F = M + 1;
  __shared__ float2 s[fft_smem_elems(M)];
  __shared__ float red[32];
  const int tid = threadIdx.x;
  int64_t seg = first_seg + blockIdx.x;
  const int c = blockIdx.y;
  int64_t x_start = seg * hop;
  int64_t out_slot = seg - first_seg;
  if (gate.d_n != nullptr) {
    // streaming (O-6): the segment that ends at the newest sample, only on updates that complete one
    const int64_t n = *gate.d_n;
    if (n < NFFT || (n % hop) != 0) return;
    x_start = (n - NFFT) % gate.ring_len;
    out_slot = (n / hop - 2) % seg_stride_out;
  }
  const float* x = strain + (int64_t)c * ld;
  const int64_t ring = gate.d_n != nullptr ? gate.ring_len : 0;

  float2 v[M / NT];
  float sum = 0.f;
#pragma unroll
  for (int i = 0; i < M / NT; ++i) {
    const int n = tid + i * NT;
    int64_t i0 = x_start + 2 * n, i1 = i0 + 1;
    if (ring) { if (i0 >= ring) i0 -= ring; if (i1 >= ring) i1 -= ring; }
    v[i].x = x[i0] * scale;
    v[i].y = x[i1] * scale;
    sum += v[i].x + v[i].y;
  }
  // block reduction of the segment sum (detrend = 'constant', reading A1)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if ((tid & 31) == 0) red[tid >> 5] = sum;
  __syncthreads();
  float tot = 0.f;
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) tot += red[w];
  const float mean = tot * (1.0f / NFFT);
#pragma unroll
  for (int i = 0; i < M / NT; ++i) {
    const int n = tid + i * NT;
    const float w0 = 0.5f - 0.5f * tw[(2 * n) * (AF_TW_N / NFFT)].x;       // periodic Hann
    const float w1 = 0.5f - 0.5f * tw[(2 * n + 1) * (AF_TW_N / NFFT)].x;
    s[fft_pad(n)] = make_float2((v[i].x - mean) * w0, (v[i].y - mean) * w1);
  }
  __syncthreads();
  fft_smem<float2, M, NT>(s, tw, tid);

  float* out = pgram + ((int64_t)c * seg_stride_out + out_slot) * F;
  for (int k = tid; k <= M / 2; k += NT) {
    const float2 zk = s[fft_pad(k)];
    const float2 zm = s[fft_pad((M - k) & (M - 1))];
    const float2 e = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    const float2 o = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));   // -i (zk - conj zm)/2
    const float2 wo = cmul(tw[k * (AF_TW_N / NFFT)], o);
    const float2 xk = cadd(e, wo), xm = csub(e, wo);      // X[k], conj(X[M-k])
    const float pk = (xk.x * xk.x + xk.y * xk.y) * norm;
    const float pm = (xm.x * xm.x + xm.y * xm.y) * norm;
    if (k == 0) { out[0] = pk; out[M] = pm; }
    else if (k == M / 2) { out[k] = 2.f * pk; }
    else { out[k] = 2.f * pk; out[M - k] = 2.f * pm; }
  }
}

// PSD of epoch e = mean of n_avg consecutive periodograms starting at segment e*seg_step.
__global__ void psd_mean_kernel(const float* __restrict__ pgram, int64_t n_seg_total, int64_t seg_step, int n_avg,
                                int F, int C, float* __restrict__ psd, StreamGate gate) {
  if (gate.d_n != nullptr && !gate.psd_due()) return;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t e = blockIdx.y;
  const int c = blockIdx.z;
  if (k >= F) return;
  const float* p = pgram + ((int64_t)c * n_seg_total + e * seg_step) * F + k;
  double acc = 0.0;
  for (int j = 0; j < n_avg; ++j) acc += (double)p[(int64_t)j * F];
  psd[((int64_t)e * C + c) * F + k] = (float)(acc / n_avg);
}

// NEXT-3 variant: per-bin MEDIAN of the n_avg periodograms (n_avg <= 255) times 1 / median_bias(n_avg) (computed on the
// host in double).  One thread per bin: insertion sort of its column in local memory; even n_avg averages the two
// middle values.  The order in which the periodograms sit in the ring does not matter.
__global__ void psd_median_kernel(const float* __restrict__ pgram, int64_t n_seg_total, int64_t seg_step, int n_avg,
                                  int F, int C, float inv_bias, float* __restrict__ psd, StreamGate gate) {
  if (gate.d_n != nullptr && !gate.psd_due()) return;
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t e = blockIdx.y;
  const int c = blockIdx.z;
  if (k >= F) return;
  const float* p = pgram + ((int64_t)c * n_seg_total + e * seg_step) * F + k;
  float v[255];
  for (int j = 0; j < n_avg; ++j) {
    const float x = p[(int64_t)j * F];
    int i = j;
    while (i > 0 && v[i - 1] > x) { v[i] = v[i - 1]; --i; }
    v[i] = x;
  }
  const float med = (n_avg & 1) ? v[n_avg / 2] : 0.5f * (v[n_avg / 2 - 1] + v[n_avg / 2]);
  psd[((int64_t)e * C + c) * F + k] = med * inv_bias;
}

// --------------------------------------------------------------------------------------------------
// Filter design (double).  One CTA per (epoch, channel).
//   A[k] = 1/sqrt(P_d[k] fs/2) in band; g = irfft_{N_d}(A) (A real & even -> one complex FFT, real part);
//   h[j] = g[|j|] cos^2(pi j / L); H = rfft_{N_os}(h placed circularly) (real) ; stored as H / (N_os/2).
// --------------------------------------------------------------------------------------------------
template <int ND>
__global__ void __launch_bounds__(512)
filter_design_kernel(const float* __restrict__ psd, int F_w, int C, double fs, double f_lo, double f_hi, int L,
                     const double2* __restrict__ tw, float* __restrict__ H_out, float* __restrict__ taps_out,
                     StreamGate gate) {
  if (gate.d_n != nullptr) {
    if (!gate.psd_due()) return;
    if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0) *gate.d_has_filter = 1;
  }
  constexpr int NT = 512;
  constexpr int NOS = AF_NOS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double2* s = reinterpret_cast<double2*>(smem_raw);            // fft_smem_elems(8192) double2
  double* g = reinterpret_cast<double*>(s + fft_smem_elems(NOS)); // L/2 + 1 doubles
  const int tid = threadIdx.x;
  const int64_t ec = (int64_t)blockIdx.x * C + blockIdx.y;
  const float* P = psd + ec * F_w;
  const int nfft_w = 2 * (F_w - 1);
  const int half = L / 2;

  for (int k = tid; k <= ND / 2; k += NT) {
    // linear interpolation of the PSD at f = k fs / ND  (position k * nfft_w / ND in Welch bins)
    const int64_t num = (int64_t)k * nfft_w;
    const int i = (int)(num / ND);
    const double frac = (double)(num - (int64_t)i * ND) / ND;
    const double pd = (i >= F_w - 1) ? (double)P[F_w - 1] : (1.0 - frac) * (double)P[i] + frac * (double)P[i + 1];
    const double f = k * fs / ND;
    const double a = (f >= f_lo && f <= f_hi) ? 1.0 / sqrt(pd * fs * 0.5) : 0.0;
    s[fft_pad(k)] = make_double2(a, 0.0);
    if (k > 0 && k < ND / 2) s[fft_pad(ND - k)] = make_double2(a, 0.0);
  }
  __syncthreads();
  fft_smem<double2, ND, NT>(s, tw, tid);
  for (int n = tid; n <= half; n += NT) g[n] = s[fft_pad(n)].x / ND;
  __syncthreads();
  for (int n = tid; n < NOS; n += NT) {
    int j = (n <= NOS / 2) ? n : n - NOS;            // circular placement of lag j
    const int aj = j < 0 ? -j : j;
    double h = 0.0;
    if (aj < half) { const double cw = cospi((double)aj / L); h = g[aj] * cw * cw; }
    s[fft_pad(n)] = make_double2(h, 0.0);
  }
  if (taps_out != nullptr) {
    float* t = taps_out + ec * (L + 1);
    for (int n = tid; n <= L; n += NT) {
      const int aj = n < half ? half - n : n - half;
      double h = 0.0;
      if (aj < half) { const double cw = cospi((double)aj / L); h = g[aj] * cw * cw; }
      t[n] = (float)h;
    }
  }
  __syncthreads();
  fft_smem<double2, NOS, NT>(s, tw, tid);
  float* Ho = H_out + ec * (NOS / 2 + 1);
  for (int k = tid; k <= NOS / 2; k += NT) Ho[k] = (float)(s[fft_pad(k)].x * (2.0 / NOS));
}

// --------------------------------------------------------------------------------------------------
// host launchers
// --------------------------------------------------------------------------------------------------
aframe_status af_launch_welch_periodograms(aframe_ctx* ctx, const float* d_strain, int64_t ld, int64_t first_seg,
                                           int64_t n_seg, float* d_pgram, const StreamGate* gate_in) {
  if (n_seg <= 0) return AFRAME_OK;
  if (!gate_in && first_seg == 0 && af_welch_pair_applicable(ctx, n_seg)) return af_launch_welch_pairs(ctx, d_strain, ld, n_seg, d_pgram);
  StreamGate gate = gate_in ? *gate_in : StreamGate();
  if (gate_in) { first_seg = 0; }
  const aframe_config& cfg = ctx->cfg;
  const int nfft = cfg.welch_nfft;
  const float scale = ldexpf(1.0f, cfg.strain_scale_log2);
  const double sum_w2 = 0.375 * nfft;                 // sum of the periodic Hann window squared
  const float norm = (float)(1.0 / (cfg.fs * sum_w2));
  dim3 grid((unsigned)(gate_in ? 1 : n_seg), (unsigned)af_nch(ctx));
  af_prof_begin(ctx, AFRAME_PROF_WELCH);
#define AF_WELCH_CASE(N)                                                                                            \
  case N:                                                                                                           \
    welch_periodogram_kernel<N><<<grid, N / 32, 0, ctx->stream>>>(d_strain, ld, cfg.welch_hop, first_seg, n_seg,    \
                                                                  scale, norm, ctx->d_tw32, d_pgram, gate);         \
    break;
  switch (nfft) {
    AF_WELCH_CASE(1024) AF_WELCH_CASE(2048) AF_WELCH_CASE(4096) AF_WELCH_CASE(8192)
    default: return af_fail(ctx, AFRAME_EINVAL, "welch_nfft must be a power of two in 1024..8192");
  }
#undef AF_WELCH_CASE
  af_prof_end(ctx, AFRAME_PROF_WELCH, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

aframe_status af_launch_psd_mean(aframe_ctx* ctx, const float* d_pgram, int64_t n_seg_total, int64_t seg_step,
                                 int64_t n_epochs, int64_t n_avg, float* d_psd, const StreamGate* gate_in) {
  StreamGate gate = gate_in ? *gate_in : StreamGate();
  if (n_epochs <= 0) return AFRAME_OK;
  const int F = ctx->cfg.welch_nfft / 2 + 1;
  dim3 grid((F + 127) / 128, (unsigned)n_epochs, (unsigned)af_nch(ctx));
  af_prof_begin(ctx, AFRAME_PROF_WELCH);
  if (ctx->cfg.welch_average == 1) {
    if (n_avg > 255) return af_fail(ctx, AFRAME_EUNSUPPORTED, "median Welch: more than 255 segments");
    const int64_t m = (n_avg & 1) ? n_avg : n_avg - 1;
    double bias = 0.0;                                 // sum_{i=1}^{m} (-1)^(i+1) / i
    for (int64_t i = 1; i <= m; ++i) bias += ((i & 1) ? 1.0 : -1.0) / (double)i;
    psd_median_kernel<<<grid, 128, 0, ctx->stream>>>(d_pgram, n_seg_total, seg_step, (int)n_avg, F, af_nch(ctx),
                                                     (float)(1.0 / bias), d_psd, gate);
  } else
    psd_mean_kernel<<<grid, 128, 0, ctx->stream>>>(d_pgram, n_seg_total, seg_step, (int)n_avg, F, af_nch(ctx), d_psd, gate);
  af_prof_end(ctx, AFRAME_PROF_WELCH, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

static size_t filter_design_smem(int L) { return sizeof(double2) * fft_smem_elems(AF_NOS) + sizeof(double) * (L / 2 + 1); }

aframe_status af_launch_filter_design(aframe_ctx* ctx, const float* d_psd, int64_t n_epochs, float* d_H, float* d_taps,
                                      const StreamGate* gate_in) {
  if (n_epochs <= 0) return AFRAME_OK;
  StreamGate gate = gate_in ? *gate_in : StreamGate();
  const aframe_config& cfg = ctx->cfg;
  const size_t smem = filter_design_smem(cfg.filter_len);
  dim3 grid((unsigned)n_epochs, (unsigned)af_nch(ctx));
  const int F_w = cfg.welch_nfft / 2 + 1;
  af_prof_begin(ctx, AFRAME_PROF_DESIGN);
#define AF_FD_CASE(N)                                                                                                \
  case N: {                                                                                                          \
    static std::atomic<uint64_t> attr_done{0};           /* bit d: set on device d (the attribute is per device) */  \
    const uint64_t bit = 1ull << (ctx->device & 63);                                                                 \
    if (!(attr_done.load(std::memory_order_acquire) & bit)) {                                                        \
      AF_CUDA(ctx, cudaFuncSetAttribute(filter_design_kernel<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
      attr_done.fetch_or(bit, std::memory_order_release);                                                            \
    }                                                                                                                \
    filter_design_kernel<N><<<grid, 512, smem, ctx->stream>>>(d_psd, F_w, af_nch(ctx), cfg.fs, cfg.f_lo, cfg.f_hi, \
                                                             cfg.filter_len, ctx->d_tw64, d_H, d_taps, gate);        \
  } break;
  switch (cfg.n_design) {
    AF_FD_CASE(1024) AF_FD_CASE(2048) AF_FD_CASE(4096) AF_FD_CASE(8192)
    default: return af_fail(ctx, AFRAME_EINVAL, "n_design must be a power of two in 1024..8192");
  }
#undef AF_FD_CASE
  af_prof_end(ctx, AFRAME_PROF_DESIGN, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
