// Shared host/device helpers of the aframe B200 library (not shared with oracle/).
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

#include "../../include/aframe.h"

#define AF_MAX_CH 8
#if defined(__GNUC__)
#define AF_API extern "C" __attribute__((visibility("default")))
#else
#define AF_API extern "C"
#endif

// Storage types (values of aframe_precision): fp32, bf16, fp16.
enum { AF_DT_F32 = 0, AF_DT_BF16 = 1, AF_DT_F16 = 2 };
static inline size_t af_dt_bytes(int dt) { return dt == AF_DT_F32 ? 4 : 2; }

// Weights and activations of the tensor-core path are stored as IEEE half (reading B10 of DESIGN.md: with one bf16
// rounding per stored activation the scores lose their rank order -- Spearman 0.9987 against the float64 oracle on
// configs[1], the ceiling of that format -- while fp16's three extra mantissa bits give > 0.9999 at the same bytes and
// the same tcgen05 kind::f16 rate; the instruction wants A and B in ONE format: a mixed fp16 x bf16 descriptor raises
// an illegal-instruction fault on B200).  Conversions round to nearest even and saturate at +-65504 (NaN stays NaN).
typedef __half af_act_t;
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t af_act_pack2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ float2 af_act_unpack2(uint32_t w) { return __half22float2(*reinterpret_cast<const __half2*>(&w)); }
// one element of a whitened stream / window tensor of storage type DT -> fp32
template <int DT> __device__ __forceinline__ float af_ld_as_f32(const void* p, int64_t i) {
  if (DT == AF_DT_BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[i]);
  if (DT == AF_DT_F16) return __half2float(reinterpret_cast<const __half*>(p)[i]);
  return __ldg(reinterpret_cast<const float*>(p) + i);
}
#endif

struct LayerDesc {
  int kind, c_in, c_out, k, stride, pad, relu, input_from, residual_from;
  int t_in, t_out;
};

// Folded network on the device.
struct aframe_weights {
  aframe_ctx* ctx = nullptr;
  std::vector<LayerDesc> layers;
  int in_channels = 0;
  int kernel_len = 0;
  // per conv layer (index = layer index; null for other kinds)
  std::vector<float*> d_w32;          // [k][c_in][c_out] fp32 (N contiguous) for the CUDA-core path
  std::vector<af_act_t*> d_w16;       // [k][c_out][c_in] fp16 (K-major) for the tcgen05 path
  std::vector<float*> d_bias;         // [c_out] fp32 folded bias
  std::vector<float*> d_bias_sc;      // conv whose residual is a 1x1 projection conv: its bias + the projection's (else null)
  float* d_head_w = nullptr;          // [c_in]
  float head_b = 0.f;
  int head_layer = -1;
  // NEXT-2: true GroupNorm (blob norm_kind 2): statistics per window at inference, fp32 path only
  bool live_gn = false;
  int n_groups = 0;
  float gn_eps = 0.f;
  std::vector<float*> d_gamma, d_beta;   // per conv layer [c_out] (live_gn only)
  bool tc_ok = false;                 // bf16 tensor-core path available for this table
  std::string tc_reason;
};

struct ProfSpan {
  cudaEvent_t a, b;
  int kind, launches;
};

struct Workspace {
  void* ptr = nullptr;
  size_t bytes = 0;
};

struct aframe_ctx {
  aframe_config cfg;
  cudaStream_t stream = nullptr;
  int device = 0;
  int n_sms = 148;
  char err[512];
  int64_t launches = 0;
  double tc_macs = 0.0;        // multiply-accumulates issued to the tensor cores so far (conv_tc.cu; aframe_tensor_macs)
  // tables
  float2* d_tw32 = nullptr;    // exp(-2 pi i q / 8192), q < 8192
  double2* d_tw64 = nullptr;
  // scratch
  Workspace ws_psd;            // periodograms
  Workspace ws_filt;           // PSD / H / taps per epoch
  Workspace ws_act;            // network activations
  float* d_taps_last = nullptr;   // [C][L+1] of the last aframe_whiten call
  void* encode_tiled = nullptr;   // cuTensorMapEncodeTiled entry point
  Workspace ws_white;          // whitened stream of aframe_score_timeslides
  Workspace ws_stage;          // device staging of the *_host entry points
  Workspace ws_groups;         // group sums of periodograms (aframe_whiten_rolling)
  // optional per-stage device timing (aframe_profile): CUDA-event pairs on ctx->stream
  bool prof_on = false;
  std::vector<ProfSpan> prof_spans;
  std::vector<cudaEvent_t> prof_pool;
  cudaEvent_t prof_open[AFRAME_PROF_KINDS] = {};
  float* layer_ms = nullptr;   // aframe_profile_layers: per-layer device time of the next forward (host array), else null
  void* tc_cache = nullptr;    // conv_tc.cu: cached tensor maps / launch plans of the bf16 path (af_tc_forget frees it)
  int n_ch_batch = 0;          // aframe_whiten_batch: rows (element x detector) the signal launchers treat as channels
  // objects created from this context that are still alive: aframe_destroy releases their device resources and marks
  // them dead (ctx = nullptr), after which aframe_weights_free / aframe_stream_destroy only delete the host shell
  std::vector<aframe_weights*> live_weights;
  std::vector<aframe_stream_state*> live_streams;
};

void af_weights_release(aframe_weights* w);             // device arrays of a weights object (aframe_api.cu)
void af_stream_release(aframe_stream_state* st);        // device blob and captured graphs of a stream state (stream.cu)
const aframe_weights* af_stream_weights(const aframe_stream_state* st);

// rows the Welch / design / whitening launchers run over: the configured detectors, or a training batch's B*C rows
static inline int af_nch(const aframe_ctx* ctx) { return ctx->n_ch_batch > 0 ? ctx->n_ch_batch : ctx->cfg.n_channels; }

// Stage timing: af_prof_begin records an event before the first launch of a stage, af_prof_end one after
// its last launch; aframe_profile_read sums the elapsed times per stage.  No-ops unless profiling is on.
void af_prof_begin(aframe_ctx* ctx, int kind);
void af_prof_end(aframe_ctx* ctx, int kind, int launches);

#define AF_TW_N 8192
#define AF_NOS 8192   // overlap-save block (real samples)

static inline aframe_status af_fail(aframe_ctx* ctx, aframe_status st, const char* fmt, const char* a = "") {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), fmt, a);
  return st;
}

#define AF_CUDA(ctx, call)                                                                  \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess) {                                                                \
      if (ctx) snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, \
                        #call, cudaGetErrorString(e_));                                     \
      return AFRAME_ECUDA;                                                                  \
    }                                                                                       \
  } while (0)

#define AF_LAUNCH_CHECK(ctx)                 \
  do {                                       \
    (ctx)->launches++;                       \
    AF_CUDA(ctx, cudaGetLastError());        \
  } while (0)

aframe_status af_ws_reserve(aframe_ctx* ctx, Workspace& ws, size_t bytes);

// Device-side gate of the streaming path (O-6): the update counter lives on the device so that one
// captured CUDA graph serves every update; gated kernels return at once on updates that need no work.
struct StreamGate {
  const int64_t* d_n = nullptr;   // samples received so far (after this update's append); null = ungated
  int* d_has_filter = nullptr;
  int64_t ring_len = 0;           // raw ring length in samples
  int64_t psd_len = 0, psd_update = 0;
  __host__ __device__ bool psd_due() const {
    const int64_t n = *d_n;
    return n >= psd_len && ((n - psd_len) % psd_update) == 0;
  }
};

// ---- kernels' host entry points (defined in the .cu files) ------------------------------------
aframe_status af_launch_welch_periodograms(aframe_ctx* ctx, const float* d_strain, int64_t ld, int64_t first_seg,
                                           int64_t n_seg, float* d_pgram /*[C][n_seg][F]*/, const StreamGate* gate = nullptr);
aframe_status af_launch_psd_mean(aframe_ctx* ctx, const float* d_pgram, int64_t n_seg_total, int64_t seg0_stride,
                                 int64_t n_epochs, int64_t n_avg, float* d_psd /*[n_epochs][C][F]*/, const StreamGate* gate = nullptr);
aframe_status af_launch_filter_design(aframe_ctx* ctx, const float* d_psd, int64_t n_epochs, float* d_H /*[E][C][NOS/2+1]*/,
                                      float* d_taps /*[E][C][L+1] or null*/, const StreamGate* gate = nullptr);
aframe_status af_launch_whiten_os(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                  const float* d_H, int64_t in0, int64_t out_total, int64_t epoch_len, int64_t n_epochs,
                                  void* d_out, int64_t ld_out, int out_dt);

// signal_fft64.cu: stored records with welch_nfft 4096 take two segments per transform; many epochs take group sums
bool af_welch_pair_applicable(const aframe_ctx* ctx, int64_t n_seg);
aframe_status af_launch_welch_pairs(aframe_ctx* ctx, const float* d_strain, int64_t ld, int64_t n_seg, float* d_pgram);
aframe_status af_launch_psd_mean_grouped(aframe_ctx* ctx, const float* d_pgram, int64_t n_seg_total, int64_t seg_step,
                                         int64_t n_epochs, int64_t n_avg, float* d_groups, float* d_psd);

aframe_status af_forward_fp32(aframe_ctx* ctx, const aframe_weights* w, const void* d_in, int in_dt,
                              int64_t sB, int64_t sT, const int64_t* choff, int64_t B, float* d_scores);
aframe_status af_forward_bf16(aframe_ctx* ctx, const aframe_weights* w, const void* d_in, int in_dt,
                              int64_t sB, int64_t sT, const int64_t* choff, int64_t B, float* d_scores);
aframe_status af_tc_check(aframe_ctx* ctx, aframe_weights* w);
void af_tc_forget(aframe_ctx* ctx);
