// aframe_psd_welch_static: O-1 (Welch PSD; reading A1) for callers that may not allocate device memory --
// code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// aframe_psd_welch keeps its periodograms [C][n_seg][F] in a workspace that grows with cudaMalloc on first use at a
// larger size.  This variant runs the SAME kernels (welch_pair_kernel / welch_periodogram_kernel, then psd_mean_kernel /
// psd_median_kernel) with that scratch in a file-scope device array of fixed size, so the call allocates nothing:
// no cudaMalloc / cudaFree, no allocating library routine.  Every GPU that loads the library holds the array
// (AF_STATIC_PSD_FLOATS * 4 bytes = 1.0 MiB) until the process exits.
//
// The array is shared by every call, context and stream of the process on that device and keeps the last call's
// contents.  Nothing in it has to start at zero: a call writes the n_seg periodograms of each channel before the mean /
// median kernel reads exactly those (the launches are ordered on the context's stream).  Two calls that overlap on the
// GPU (different streams, or different contexts on different streams) race on it: serialise them.
#include <atomic>
#include "common.cuh"

// periodograms of up to 64 Welch segments of two detectors at welch_nfft 4096 (the 64 s PSD of P:172 is 63 segments)
#define AF_STATIC_PSD_FLOATS (2 * 64 * 2049)

static __device__ __align__(256) float g_psd_static_scratch[AF_STATIC_PSD_FLOATS];

// In host code the array's name is a host-side stand-in, not a device address: the kernels get the address
// cudaGetSymbolAddress returns, looked up once per device with that device current.
static constexpr int AF_STATIC_MAX_DEVICES = 64;
static std::atomic<float*> g_psd_static_ptr[AF_STATIC_MAX_DEVICES];

static aframe_status psd_static_address(aframe_ctx* ctx, float** out) {
  int dev = -1;
  AF_CUDA(ctx, cudaGetDevice(&dev));
  if (dev != ctx->device) return af_fail(ctx, AFRAME_ESTATE, "aframe_psd_welch_static: the context's device is not the current device");
  if (dev < 0 || dev >= AF_STATIC_MAX_DEVICES) return af_fail(ctx, AFRAME_EUNSUPPORTED, "aframe_psd_welch_static: device ordinal above 63");
  float* p = g_psd_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    void* sym = nullptr;
    AF_CUDA(ctx, cudaGetSymbolAddress(&sym, g_psd_static_scratch));
    if (!sym) return af_fail(ctx, AFRAME_ECUDA, "aframe_psd_welch_static: cudaGetSymbolAddress returned a null address");
    p = static_cast<float*>(sym);
    g_psd_static_ptr[dev].store(p, std::memory_order_release);   // (two racing threads store the same value)
  }
  *out = p;
  return AFRAME_OK;
}

AF_API int64_t aframe_psd_welch_static_max_floats(void) { return AF_STATIC_PSD_FLOATS; }

AF_API aframe_status aframe_psd_welch_static(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                             float* d_psd) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_strain || !d_psd) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  const aframe_config& cfg = ctx->cfg;
  if (n_samples < cfg.welch_nfft || ld < n_samples) return af_fail(ctx, AFRAME_ESHAPE, "n_samples < welch_nfft or ld < n_samples");
  const int64_t n_seg = (n_samples - cfg.welch_nfft) / cfg.welch_hop + 1;
  const int F = cfg.welch_nfft / 2 + 1;
  const int64_t need = (int64_t)cfg.n_channels * n_seg * F;
  if (need > AF_STATIC_PSD_FLOATS) {
    snprintf(ctx->err, sizeof(ctx->err),
             "aframe_psd_welch_static: n_channels * segments * (welch_nfft / 2 + 1) = %lld floats exceeds the static scratch of %d "
             "(use aframe_psd_welch, which allocates)", (long long)need, AF_STATIC_PSD_FLOATS);
    return AFRAME_ESHAPE;
  }
  float* pg = nullptr;
  aframe_status st = psd_static_address(ctx, &pg);
  if (st != AFRAME_OK) return st;
  st = af_launch_welch_periodograms(ctx, d_strain, ld, 0, n_seg, pg);
  if (st != AFRAME_OK) return st;
  return af_launch_psd_mean(ctx, pg, n_seg, 0, 1, n_seg, d_psd);
}
