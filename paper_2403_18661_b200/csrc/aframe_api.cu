// C-ABI entry points (include/aframe.h): context, PSD, whitening, weights, forward.
// Host logic only; every step of the path runs in the kernels of the other translation units.
#include <math.h>
#include <string.h>
#include <new>

#include "common.cuh"
#include "net_plan.h"

static const char* kNoCtx = "no context";

AF_API aframe_status aframe_config_default(aframe_config* cfg) {
  if (!cfg) return AFRAME_EINVAL;
  memset(cfg, 0, sizeof(*cfg));
  cfg->size = (uint32_t)sizeof(aframe_config);
  cfg->n_channels = 2;
  cfg->fs = 2048.0;
  cfg->welch_nfft = 4096;
  cfg->welch_hop = 2048;
  cfg->filter_len = 2048;
  cfg->n_design = 8192;
  cfg->f_lo = 20.0;
  cfg->f_hi = 1000.0;
  cfg->kernel_len = 3072;
  cfg->stride = 128;
  cfg->psd_len = 131072;
  cfg->psd_update = 16384;
  cfg->strain_scale_log2 = 70;
  cfg->precision = AFRAME_F16;
  return AFRAME_OK;
}

static bool is_pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }

aframe_status af_ws_reserve(aframe_ctx* ctx, Workspace& ws, size_t bytes) {
  if (bytes <= ws.bytes) return AFRAME_OK;
  // growing: wait for queued work that may still read the old buffer, then replace it
  AF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  if (ws.ptr) cudaFree(ws.ptr);
  ws.ptr = nullptr; ws.bytes = 0;
  const size_t want = bytes + bytes / 8;
  cudaError_t e = cudaMalloc(&ws.ptr, want);
  if (e != cudaSuccess) {
    cudaGetLastError();
    e = cudaMalloc(&ws.ptr, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); ws.ptr = nullptr; return af_fail(ctx, AFRAME_ENOMEM, "device workspace allocation failed"); }
    ws.bytes = bytes;
  } else {
    ws.bytes = want;
  }
  return AFRAME_OK;
}

AF_API aframe_status aframe_create(const aframe_config* cfg, void* cuda_stream, aframe_ctx** out) {
  if (!cfg || !out) return AFRAME_EINVAL;
  *out = nullptr;
  if (cfg->size != sizeof(aframe_config)) return AFRAME_EINVAL;
  if (cfg->n_channels < 1 || cfg->n_channels > AF_MAX_CH) return AFRAME_EINVAL;
  if (!(cfg->fs > 0)) return AFRAME_EINVAL;
  if (!is_pow2(cfg->welch_nfft) || cfg->welch_nfft < 1024 || cfg->welch_nfft > 8192) return AFRAME_EINVAL;
  if (cfg->welch_hop * 2 != cfg->welch_nfft) return AFRAME_EINVAL;
  if (!is_pow2(cfg->n_design) || cfg->n_design < 1024 || cfg->n_design > 8192) return AFRAME_EINVAL;
  if (cfg->filter_len < 2 || (cfg->filter_len & 1) || cfg->filter_len > AF_NOS / 2) return AFRAME_EINVAL;
  if (cfg->filter_len > cfg->n_design) return AFRAME_ESHAPE;
  if (!(cfg->f_lo >= 0) || !(cfg->f_hi > cfg->f_lo) || cfg->f_hi > cfg->fs / 2) return AFRAME_EINVAL;
  if (cfg->kernel_len < 1 || cfg->stride < 1) return AFRAME_EINVAL;
  if (cfg->psd_len < cfg->welch_nfft || cfg->psd_len % cfg->welch_hop) return AFRAME_ESHAPE;
  if (cfg->psd_update < 1 || cfg->psd_update % cfg->welch_hop || cfg->psd_update % cfg->stride) return AFRAME_ESHAPE;
  if (cfg->psd_len % cfg->stride) return AFRAME_ESHAPE;
  if (cfg->strain_scale_log2 < -120 || cfg->strain_scale_log2 > 120) return AFRAME_EINVAL;
  if (cfg->precision == AFRAME_BF16) return AFRAME_EUNSUPPORTED;   // bf16 storage cannot meet the rank tolerance (aframe.h)
  if (cfg->precision != AFRAME_FP32 && cfg->precision != AFRAME_F16) return AFRAME_EINVAL;
  if ((cfg->welch_average != 0 && cfg->welch_average != 1) || cfg->stream_full_forward < 0 || cfg->stream_full_forward > 2) return AFRAME_EINVAL;
  if (cfg->welch_average == 1 && (cfg->psd_len - cfg->welch_nfft) / cfg->welch_hop + 1 > 255) return AFRAME_EUNSUPPORTED;

  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return AFRAME_EUNSUPPORTED; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cudaGetLastError(); return AFRAME_EUNSUPPORTED; }
  if (prop.major != 10) return AFRAME_EUNSUPPORTED;   // sm_100a only: no fallback path exists

  aframe_ctx* ctx = new (std::nothrow) aframe_ctx();
  if (!ctx) return AFRAME_ENOMEM;
  ctx->cfg = *cfg;
  ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  ctx->device = dev;
  ctx->n_sms = prop.multiProcessorCount;
  ctx->err[0] = 0;

  std::vector<float2> t32(AF_TW_N);
  std::vector<double2> t64(AF_TW_N);
  for (int q = 0; q < AF_TW_N; ++q) {
    // exact octant symmetry is not needed; cos/sin in double of the reduced angle
    const double ang = -2.0 * M_PI * (double)q / AF_TW_N;
    t64[q] = make_double2(cos(ang), sin(ang));
    t32[q] = make_float2((float)t64[q].x, (float)t64[q].y);
  }
  t64[0] = make_double2(1.0, 0.0);            t32[0] = make_float2(1.f, 0.f);
  t64[AF_TW_N / 4] = make_double2(0.0, -1.0); t32[AF_TW_N / 4] = make_float2(0.f, -1.f);
  t64[AF_TW_N / 2] = make_double2(-1.0, 0.0); t32[AF_TW_N / 2] = make_float2(-1.f, 0.f);
  t64[3 * AF_TW_N / 4] = make_double2(0.0, 1.0); t32[3 * AF_TW_N / 4] = make_float2(0.f, 1.f);
  aframe_status st = AFRAME_OK;
  do {
    if (cudaMalloc(&ctx->d_tw32, sizeof(float2) * AF_TW_N) != cudaSuccess ||
        cudaMalloc(&ctx->d_tw64, sizeof(double2) * AF_TW_N) != cudaSuccess ||
        cudaMalloc(&ctx->d_taps_last, sizeof(float) * cfg->n_channels * (cfg->filter_len + 1)) != cudaSuccess) {
      st = AFRAME_ENOMEM; break;
    }
    if (cudaMemcpy(ctx->d_tw32, t32.data(), sizeof(float2) * AF_TW_N, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(ctx->d_tw64, t64.data(), sizeof(double2) * AF_TW_N, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(ctx->d_taps_last, 0, sizeof(float) * cfg->n_channels * (cfg->filter_len + 1)) != cudaSuccess) {
      st = AFRAME_ECUDA; break;
    }
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ctx->encode_tiled, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      ctx->encode_tiled = nullptr;   // the tensor-core path will report EUNSUPPORTED
    }
    if (cudaDeviceSynchronize() != cudaSuccess) { st = AFRAME_ECUDA; break; }
  } while (0);
  if (st != AFRAME_OK) { cudaGetLastError(); aframe_destroy(ctx); return st; }
  *out = ctx;
  return AFRAME_OK;
}

AF_API void aframe_destroy(aframe_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
  // children that outlive their context are released here and left as dead shells (aframe.h, "Lifetime")
  for (aframe_stream_state* st : ctx->live_streams) af_stream_release(st);
  ctx->live_streams.clear();
  for (aframe_weights* w : ctx->live_weights) { af_weights_release(w); w->ctx = nullptr; }
  ctx->live_weights.clear();
  af_tc_forget(ctx);
  cudaFree(ctx->d_tw32); cudaFree(ctx->d_tw64); cudaFree(ctx->d_taps_last);
  cudaFree(ctx->ws_psd.ptr); cudaFree(ctx->ws_filt.ptr); cudaFree(ctx->ws_act.ptr);
  cudaFree(ctx->ws_white.ptr); cudaFree(ctx->ws_stage.ptr); cudaFree(ctx->ws_groups.ptr);
  for (ProfSpan& s : ctx->prof_spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  for (cudaEvent_t e : ctx->prof_pool) cudaEventDestroy(e);
  for (int k = 0; k < AFRAME_PROF_KINDS; ++k) if (ctx->prof_open[k]) cudaEventDestroy(ctx->prof_open[k]);
  cudaGetLastError();
  delete ctx;
}

AF_API const char* aframe_last_error(const aframe_ctx* ctx) { return ctx ? ctx->err : kNoCtx; }
AF_API int64_t aframe_launch_count(const aframe_ctx* ctx) { return ctx ? ctx->launches : 0; }
AF_API double aframe_tensor_macs(const aframe_ctx* ctx) { return ctx ? ctx->tc_macs : 0.0; }

// ---- O-1 ------------------------------------------------------------------------------------------
AF_API aframe_status aframe_psd_welch(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                          float* d_psd) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_strain || !d_psd) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  const aframe_config& cfg = ctx->cfg;
  if (n_samples < cfg.welch_nfft || ld < n_samples) return af_fail(ctx, AFRAME_ESHAPE, "n_samples < welch_nfft or ld < n_samples");
  const int64_t n_seg = (n_samples - cfg.welch_nfft) / cfg.welch_hop + 1;
  const int F = cfg.welch_nfft / 2 + 1;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_psd, sizeof(float) * (size_t)cfg.n_channels * n_seg * F);
  if (st != AFRAME_OK) return st;
  float* pg = reinterpret_cast<float*>(ctx->ws_psd.ptr);
  st = af_launch_welch_periodograms(ctx, d_strain, ld, 0, n_seg, pg);
  if (st != AFRAME_OK) return st;
  return af_launch_psd_mean(ctx, pg, n_seg, 0, 1, n_seg, d_psd);
}

// ---- O-2 / O-3 ------------------------------------------------------------------------------------
AF_API aframe_status aframe_whiten(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                       const float* d_psd, void* d_out, int64_t ld_out, aframe_precision out_dtype) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_strain || !d_psd || !d_out) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (out_dtype != AFRAME_FP32 && out_dtype != AFRAME_BF16 && out_dtype != AFRAME_F16) return af_fail(ctx, AFRAME_EINVAL, "bad out_dtype");
  const aframe_config& cfg = ctx->cfg;
  if (n_samples < 0 || ld < n_samples) return af_fail(ctx, AFRAME_ESHAPE, "ld < n_samples");
  const int64_t n_out = n_samples - cfg.filter_len;
  if (n_out > 0 && ld_out < n_out) return af_fail(ctx, AFRAME_ESHAPE, "ld_out < n_samples - filter_len");
  aframe_status st = af_ws_reserve(ctx, ctx->ws_filt, sizeof(float) * (size_t)cfg.n_channels * (AF_NOS / 2 + 1));
  if (st != AFRAME_OK) return st;
  float* H = reinterpret_cast<float*>(ctx->ws_filt.ptr);
  st = af_launch_filter_design(ctx, d_psd, 1, H, ctx->d_taps_last);
  if (st != AFRAME_OK) return st;
  if (n_out <= 0) return AFRAME_OK;
  return af_launch_whiten_os(ctx, d_strain, n_samples, ld, H, 0, n_out, n_out, 1, d_out, ld_out, (int)out_dtype);
}

// ---- NEXT-4: training-time whitening batch --------------------------------------------------
AF_API aframe_status aframe_whiten_batch(aframe_ctx* ctx, const float* d_strain, int64_t n_batch, int64_t n_samples,
                                             int64_t n_psd, void* d_out, aframe_precision out_dtype) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_strain || !d_out) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (out_dtype != AFRAME_FP32 && out_dtype != AFRAME_BF16 && out_dtype != AFRAME_F16) return af_fail(ctx, AFRAME_EINVAL, "bad out_dtype");
  const aframe_config& cfg = ctx->cfg;
  if (n_batch < 1) return af_fail(ctx, AFRAME_EINVAL, "n_batch < 1");
  const int64_t rows = n_batch * cfg.n_channels;
  const int64_t n_w = n_samples - n_psd, n_out = n_w - cfg.filter_len;
  if (n_psd < cfg.welch_nfft || n_out <= 0 || rows > 65535)
    return af_fail(ctx, AFRAME_ESHAPE, "whiten_batch: n_psd < welch_nfft, n_samples - n_psd <= filter_len, or n_batch * C > 65535");
  const int64_t n_seg = (n_psd - cfg.welch_nfft) / cfg.welch_hop + 1;
  const int F = cfg.welch_nfft / 2 + 1;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_psd, sizeof(float) * (size_t)rows * n_seg * F);
  if (st != AFRAME_OK) return st;
  st = af_ws_reserve(ctx, ctx->ws_filt, sizeof(float) * (size_t)rows * (F + AF_NOS / 2 + 1));
  if (st != AFRAME_OK) return st;
  float* pg = reinterpret_cast<float*>(ctx->ws_psd.ptr);
  float* psd = reinterpret_cast<float*>(ctx->ws_filt.ptr);
  float* H = psd + (size_t)rows * F;
  ctx->n_ch_batch = (int)rows;               // the launchers below treat every (element, detector) row as a channel
  st = af_launch_welch_periodograms(ctx, d_strain, n_samples, 0, n_seg, pg);
  if (st == AFRAME_OK) st = af_launch_psd_mean(ctx, pg, n_seg, 0, 1, n_seg, psd);
  if (st == AFRAME_OK) st = af_launch_filter_design(ctx, psd, 1, H, nullptr);
  if (st == AFRAME_OK)
    st = af_launch_whiten_os(ctx, d_strain + n_psd, n_w, n_samples, H, 0, n_out, n_out, 1, d_out, n_out, (int)out_dtype);
  ctx->n_ch_batch = 0;
  return st;
}

AF_API aframe_status aframe_filter_taps(aframe_ctx* ctx, float* d_taps) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_taps) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  AF_CUDA(ctx, cudaMemcpyAsync(d_taps, ctx->d_taps_last, sizeof(float) * ctx->cfg.n_channels * (ctx->cfg.filter_len + 1),
                               cudaMemcpyDeviceToDevice, ctx->stream));
  return AFRAME_OK;
}

// ---- O-6 offline ----------------------------------------------------------------------------------
AF_API aframe_status aframe_whiten_rolling(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                               void* d_out, int64_t ld_out, aframe_precision out_dtype, int64_t* h_n_out) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_strain || !d_out || !h_n_out) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (out_dtype != AFRAME_FP32 && out_dtype != AFRAME_BF16 && out_dtype != AFRAME_F16) return af_fail(ctx, AFRAME_EINVAL, "bad out_dtype");
  const aframe_config& cfg = ctx->cfg;
  *h_n_out = 0;
  if (n_samples < 0 || ld < n_samples) return af_fail(ctx, AFRAME_ESHAPE, "ld < n_samples");
  const int64_t n_eff = (n_samples / cfg.stride) * cfg.stride;
  if (n_eff < cfg.psd_len) return AFRAME_OK;
  const int64_t half = cfg.filter_len / 2;
  const int64_t m0 = cfg.psd_len - cfg.stride - half;          // first whitened raw index (reading C1)
  if (m0 - half < 0) return af_fail(ctx, AFRAME_ESHAPE, "psd_len < stride + filter_len");
  const int64_t n_out = n_eff - half - m0;
  if (ld_out < n_out) return af_fail(ctx, AFRAME_ESHAPE, "ld_out too small for the whitened output");
  const int64_t n_epochs = (n_eff - cfg.psd_len) / cfg.psd_update + 1;
  const int64_t seg_total = (n_eff - cfg.welch_nfft) / cfg.welch_hop + 1;
  const int64_t n_avg = (cfg.psd_len - cfg.welch_nfft) / cfg.welch_hop + 1;
  const int64_t seg_step = cfg.psd_update / cfg.welch_hop;
  const int F = cfg.welch_nfft / 2 + 1;
  const int C = cfg.n_channels;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_psd, sizeof(float) * (size_t)C * seg_total * F);
  if (st != AFRAME_OK) return st;
  const size_t psd_bytes = sizeof(float) * (size_t)n_epochs * C * F;
  const size_t H_bytes = sizeof(float) * (size_t)n_epochs * C * (AF_NOS / 2 + 1);
  st = af_ws_reserve(ctx, ctx->ws_filt, psd_bytes + H_bytes);
  if (st != AFRAME_OK) return st;
  float* pg = reinterpret_cast<float*>(ctx->ws_psd.ptr);
  float* psd = reinterpret_cast<float*>(ctx->ws_filt.ptr);
  float* H = reinterpret_cast<float*>(reinterpret_cast<char*>(ctx->ws_filt.ptr) + psd_bytes);
  st = af_launch_welch_periodograms(ctx, d_strain, ld, 0, seg_total, pg);
  if (st != AFRAME_OK) return st;
  if (cfg.welch_average == 0 && seg_step >= 2 && n_avg >= 2 * seg_step && n_epochs >= 8) {
    // consecutive epochs share all but seg_step of their n_avg periodograms: sum them in groups of seg_step once
    st = af_ws_reserve(ctx, ctx->ws_groups, 2 * sizeof(float) * (size_t)C * (seg_total / seg_step) * F);   // group sums + their first step - 1 terms
    if (st != AFRAME_OK) return st;
    st = af_launch_psd_mean_grouped(ctx, pg, seg_total, seg_step, n_epochs, n_avg, reinterpret_cast<float*>(ctx->ws_groups.ptr), psd);
  } else {
    st = af_launch_psd_mean(ctx, pg, seg_total, seg_step, n_epochs, n_avg, psd);
  }
  if (st != AFRAME_OK) return st;
  st = af_launch_filter_design(ctx, psd, n_epochs, H, nullptr);
  if (st != AFRAME_OK) return st;
  st = af_launch_whiten_os(ctx, d_strain, n_samples, ld, H, m0 - half, n_out, cfg.psd_update, n_epochs, d_out, ld_out,
                           (int)out_dtype);
  if (st != AFRAME_OK) return st;
  *h_n_out = n_out;
  return AFRAME_OK;
}

// ---- weights --------------------------------------------------------------------------------------
void af_weights_release(aframe_weights* w) {
  for (float*& p : w->d_w32) { cudaFree(p); p = nullptr; }
  for (af_act_t*& p : w->d_w16) { cudaFree(p); p = nullptr; }
  for (float*& p : w->d_bias) { cudaFree(p); p = nullptr; }
  for (float*& p : w->d_bias_sc) { cudaFree(p); p = nullptr; }
  for (float*& p : w->d_gamma) { cudaFree(p); p = nullptr; }
  for (float*& p : w->d_beta) { cudaFree(p); p = nullptr; }
  cudaFree(w->d_head_w); w->d_head_w = nullptr;
  cudaGetLastError();
}

AF_API void aframe_weights_free(aframe_weights* w) {
  if (!w) return;
  if (aframe_ctx* ctx = w->ctx) {                     // (a dead shell, released by aframe_destroy, has no context)
    cudaStreamSynchronize(ctx->stream);
    af_tc_forget(ctx);
    // stream states built on these weights can no longer step: released, and aframe_stream_step answers AFRAME_ESTATE
    for (aframe_stream_state* st : ctx->live_streams)
      if (af_stream_weights(st) == w) af_stream_release(st);
    for (size_t i = 0; i < ctx->live_weights.size(); ++i)
      if (ctx->live_weights[i] == w) { ctx->live_weights.erase(ctx->live_weights.begin() + i); break; }
    af_weights_release(w);
  }
  delete w;
}

// Header and layer table of a version-1 blob (synthdata/weights.py): validation and shape inference on the host, no CUDA call.
// hdr receives the eight header words; *why a static description of the first problem found.
aframe_status af_parse_layer_table(const void* host_blob, size_t bytes, int kernel_len, int n_channels,
                                   std::vector<LayerDesc>& layers, uint32_t hdr[8], const char** why) {
  static const char* ok = "";
  *why = ok;
  if (bytes < 32) { *why = "weight blob shorter than its header"; return AFRAME_ESHAPE; }
  memcpy(hdr, host_blob, 32);
  if (hdr[0] != 0x57524641u || hdr[1] != 1u) { *why = "bad weight blob magic/version"; return AFRAME_EINVAL; }
  const uint32_t n_layers = hdr[2], norm_kind = hdr[3], n_groups = hdr[4], in_ch = hdr[6];
  if (n_layers == 0 || n_layers > 4096 || norm_kind > 2) { *why = "bad weight blob header"; return AFRAME_EINVAL; }
  if (norm_kind >= 1 && n_groups == 0) { *why = "group norm with zero groups"; return AFRAME_EINVAL; }
  if ((int)in_ch != n_channels) { *why = "blob in_channels != cfg.n_channels"; return AFRAME_ESHAPE; }
  if (bytes < 32 + (size_t)n_layers * 48) { *why = "weight blob shorter than its layer table"; return AFRAME_ESHAPE; }
  const int32_t* tab = reinterpret_cast<const int32_t*>(reinterpret_cast<const char*>(host_blob) + 32);
  layers.assign(n_layers, LayerDesc());
  int head_layer = -1;
  for (uint32_t i = 0; i < n_layers; ++i) {
    const int32_t* r = tab + (size_t)i * 12;
    LayerDesc& l = layers[i];
    l.kind = r[0]; l.c_in = r[1]; l.c_out = r[2]; l.k = r[3]; l.stride = r[4]; l.pad = r[5]; l.relu = r[6];
    l.input_from = r[7]; l.residual_from = r[8];
    if (l.kind < 0 || l.kind > 2 || l.c_in < 1 || l.c_out < 1 || l.k < 1 || l.stride < 1 || l.pad < 0) { *why = "layer table: bad field"; return AFRAME_ESHAPE; }
    if (l.input_from >= (int)i || l.residual_from >= (int)i || l.input_from < -1 || l.residual_from < -1) { *why = "layer table: forward reference"; return AFRAME_ESHAPE; }
    const int c_src = l.input_from < 0 ? (int)in_ch : layers[l.input_from].c_out;
    const int t_src = l.input_from < 0 ? kernel_len : layers[l.input_from].t_out;
    if (l.input_from >= 0 && layers[l.input_from].kind == 2) { *why = "layer table: input from a head"; return AFRAME_ESHAPE; }
    if (c_src != l.c_in) { *why = "layer table: c_in does not match its input"; return AFRAME_ESHAPE; }
    l.t_in = t_src;
    if (l.kind == 2) {
      l.t_out = 1;
      if (l.c_out != 1) { *why = "head must have one output"; return AFRAME_ESHAPE; }
      if (head_layer >= 0 || i != n_layers - 1) { *why = "exactly one head, as the last layer"; return AFRAME_ESHAPE; }
      head_layer = (int)i;
      continue;
    }
    if (l.t_in + 2 * l.pad < l.k) { *why = "layer table: kernel longer than its padded input"; return AFRAME_ESHAPE; }
    l.t_out = (l.t_in + 2 * l.pad - l.k) / l.stride + 1;
    if (l.kind == 1) {
      if (l.c_out != l.c_in || l.residual_from >= 0) { *why = "max-pool must keep the channel count"; return AFRAME_ESHAPE; }
      continue;
    }
    if (l.residual_from >= 0) {
      const LayerDesc& rs = layers[l.residual_from];
      if (rs.kind == 2 || rs.c_out != l.c_out || rs.t_out != l.t_out) { *why = "layer table: residual shape mismatch"; return AFRAME_ESHAPE; }
    }
    if (norm_kind >= 1 && l.c_out % (int)n_groups) { *why = "c_out not divisible by n_groups"; return AFRAME_ESHAPE; }
  }
  if (head_layer < 0) { *why = "layer table has no head"; return AFRAME_ESHAPE; }
  return AFRAME_OK;
}

AF_API aframe_status aframe_weights_load(aframe_ctx* ctx, const void* host_blob, size_t bytes, aframe_weights** out) {
  if (!ctx) return AFRAME_EINVAL;
  if (!host_blob || !out) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  *out = nullptr;
  uint32_t hd[8];
  std::vector<LayerDesc> table;
  const char* why = "";
  const aframe_status pst = af_parse_layer_table(host_blob, bytes, ctx->cfg.kernel_len, ctx->cfg.n_channels, table, hd, &why);
  if (pst != AFRAME_OK) return af_fail(ctx, pst, "%s", why);
  const uint32_t n_layers = hd[2], norm_kind = hd[3], n_groups = hd[4], in_ch = hd[6];
  float eps; memcpy(&eps, &hd[5], 4);
  const size_t pay_off = 32 + (size_t)n_layers * 48;
  const float* pay = reinterpret_cast<const float*>(reinterpret_cast<const char*>(host_blob) + pay_off);
  const size_t n_pay = (bytes - pay_off) / 4;

  aframe_weights* w = new (std::nothrow) aframe_weights();
  if (!w) return af_fail(ctx, AFRAME_ENOMEM, "host allocation failed");
  w->ctx = ctx;
  w->in_channels = (int)in_ch;
  w->kernel_len = ctx->cfg.kernel_len;
  w->layers = table;
  w->d_w32.assign(n_layers, nullptr);
  w->d_w16.assign(n_layers, nullptr);
  w->d_bias.assign(n_layers, nullptr);
  w->d_bias_sc.assign(n_layers, nullptr);
  std::vector<std::vector<float>> h_bias(n_layers);
  w->d_gamma.assign(n_layers, nullptr);
  w->d_beta.assign(n_layers, nullptr);
  w->live_gn = norm_kind == 2;
  w->n_groups = (int)n_groups;
  w->gn_eps = eps;
  aframe_status st = AFRAME_OK;
  size_t pos = 0;
  auto fail = [&](aframe_status s, const char* msg) { st = af_fail(ctx, s, msg); };
  for (uint32_t i = 0; i < n_layers && st == AFRAME_OK; ++i) {
    LayerDesc& l = w->layers[i];               // (validated, shapes inferred: af_parse_layer_table)
    if (l.kind == 2) {
      if (pos + l.c_in + 1 > n_pay) { fail(AFRAME_ESHAPE, "weight blob payload too short"); break; }
      w->head_layer = (int)i;
      w->head_b = pay[pos + l.c_in];
      if (cudaMalloc(&w->d_head_w, sizeof(float) * l.c_in) != cudaSuccess) { fail(AFRAME_ENOMEM, "device allocation failed"); break; }
      if (cudaMemcpy(w->d_head_w, pay + pos, sizeof(float) * l.c_in, cudaMemcpyHostToDevice) != cudaSuccess) { fail(AFRAME_ECUDA, "weight upload failed"); break; }
      pos += l.c_in + 1;
      continue;
    }
    if (l.kind == 1) continue;
    const int n_stat = norm_kind == 0 ? l.c_out : (norm_kind == 1 ? (int)n_groups : 0);
    const size_t nw = (size_t)l.c_out * l.c_in * l.k;
    if (pos + nw + 2 * (size_t)l.c_out + 2 * (size_t)n_stat > n_pay) { fail(AFRAME_ESHAPE, "weight blob payload too short"); break; }
    const float* W = pay + pos;
    const float* gamma = W + nw;
    const float* beta = gamma + l.c_out;
    const float* mean = beta + l.c_out;
    const float* var = mean + n_stat;
    pos += nw + 2 * (size_t)l.c_out + 2 * (size_t)n_stat;
    // fold the frozen norm (reading B6) in double: W' = a_c W, b' = beta_c - mu_g a_c
    std::vector<float> w32(nw), bias(l.c_out);
    std::vector<__half> w16(nw);
    for (int co = 0; co < l.c_out; ++co) {
      const int g = norm_kind == 0 ? co : co / (l.c_out / (int)n_groups);
      // frozen norm: fold; true GroupNorm: the conv stays as it is (the norm kernels apply gamma / beta)
      const double a = norm_kind == 2 ? 1.0 : (double)gamma[co] / sqrt((double)var[g] + (double)eps);
      bias[co] = norm_kind == 2 ? 0.f : (float)((double)beta[co] - (double)mean[g] * a);
      for (int ci = 0; ci < l.c_in; ++ci)
        for (int d = 0; d < l.k; ++d) {
          const float v = (float)((double)W[((size_t)co * l.c_in + ci) * l.k + d] * a);
          w32[((size_t)d * l.c_in + ci) * l.c_out + co] = v;                      // [k][c_in][c_out]
          w16[((size_t)d * l.c_out + co) * l.c_in + ci] = __float2half_rn(fminf(fmaxf(v, -65504.f), 65504.f));  // [k][c_out][c_in]
        }
    }
    if (cudaMalloc(&w->d_w32[i], sizeof(float) * nw) != cudaSuccess || cudaMalloc(&w->d_w16[i], 2 * nw) != cudaSuccess ||
        cudaMalloc(&w->d_bias[i], sizeof(float) * l.c_out) != cudaSuccess) { fail(AFRAME_ENOMEM, "device allocation failed"); break; }
    if (cudaMemcpy(w->d_w32[i], w32.data(), sizeof(float) * nw, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(w->d_w16[i], w16.data(), 2 * nw, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(w->d_bias[i], bias.data(), sizeof(float) * l.c_out, cudaMemcpyHostToDevice) != cudaSuccess) { fail(AFRAME_ECUDA, "weight upload failed"); break; }
    h_bias[i] = bias;
    if (norm_kind == 2) {
      if (cudaMalloc(&w->d_gamma[i], sizeof(float) * l.c_out) != cudaSuccess || cudaMalloc(&w->d_beta[i], sizeof(float) * l.c_out) != cudaSuccess) { fail(AFRAME_ENOMEM, "device allocation failed"); break; }
      if (cudaMemcpy(w->d_gamma[i], gamma, sizeof(float) * l.c_out, cudaMemcpyHostToDevice) != cudaSuccess ||
          cudaMemcpy(w->d_beta[i], beta, sizeof(float) * l.c_out, cudaMemcpyHostToDevice) != cudaSuccess) { fail(AFRAME_ECUDA, "weight upload failed"); break; }
    }
  }
  // bias of a conv with its 1x1 projection shortcut folded in (the tcgen05 path runs the projection as extra K blocks)
  for (uint32_t i = 0; i < n_layers && st == AFRAME_OK; ++i) {
    const LayerDesc& l = w->layers[i];
    if (l.kind != 0 || l.residual_from < 0) continue;
    const LayerDesc& r = w->layers[l.residual_from];
    if (r.kind != 0 || r.k != 1 || r.c_out != l.c_out) continue;
    std::vector<float> b(l.c_out);
    for (int c = 0; c < l.c_out; ++c) b[c] = h_bias[i][c] + h_bias[l.residual_from][c];
    if (cudaMalloc(&w->d_bias_sc[i], sizeof(float) * l.c_out) != cudaSuccess) { fail(AFRAME_ENOMEM, "device allocation failed"); break; }
    if (cudaMemcpy(w->d_bias_sc[i], b.data(), sizeof(float) * l.c_out, cudaMemcpyHostToDevice) != cudaSuccess) { fail(AFRAME_ECUDA, "weight upload failed"); break; }
  }
  if (st == AFRAME_OK && w->head_layer < 0) st = af_fail(ctx, AFRAME_ESHAPE, "layer table has no head");
  if (st == AFRAME_OK && pos != n_pay) st = af_fail(ctx, AFRAME_ESHAPE, "weight blob payload size mismatch");
  if (st == AFRAME_OK && cudaDeviceSynchronize() != cudaSuccess) st = af_fail(ctx, AFRAME_ECUDA, "sync after weight upload failed");
  if (st != AFRAME_OK) { cudaGetLastError(); af_weights_release(w); delete w; return st; }
  af_tc_check(ctx, w);
  ctx->live_weights.push_back(w);
  *out = w;
  return AFRAME_OK;
}

// ---- O-5 ------------------------------------------------------------------------------------------
static aframe_status forward_common(aframe_ctx* ctx, const aframe_weights* w, const void* d_in, int in_dt, int64_t sB,
                                    const int64_t* choff, int64_t B, float* d_scores) {
  if (w->ctx != ctx) return af_fail(ctx, AFRAME_ESTATE, "weights belong to another context");
  if (ctx->cfg.precision == AFRAME_F16) {
    if (!w->tc_ok) return af_fail(ctx, AFRAME_EUNSUPPORTED, "fp16 tensor-core path unavailable: %s", w->tc_reason.c_str());
    return af_forward_bf16(ctx, w, d_in, in_dt, sB, 1, choff, B, d_scores);
  }
  return af_forward_fp32(ctx, w, d_in, in_dt, sB, 1, choff, B, d_scores);
}

AF_API aframe_status aframe_forward(aframe_ctx* ctx, const aframe_weights* w, const float* d_windows, int64_t B,
                                        float* d_scores) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !d_windows || !d_scores) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (B <= 0) return af_fail(ctx, AFRAME_EINVAL, "B must be positive");
  int64_t choff[AF_MAX_CH] = {0};
  for (int c = 0; c < ctx->cfg.n_channels; ++c) choff[c] = (int64_t)c * ctx->cfg.kernel_len;
  return forward_common(ctx, w, d_windows, 0, (int64_t)ctx->cfg.n_channels * ctx->cfg.kernel_len, choff, B, d_scores);
}

AF_API aframe_status aframe_forward_strided(aframe_ctx* ctx, const aframe_weights* w, const void* d_white,
                                                aframe_precision dtype, int64_t ld, int64_t first,
                                                const int64_t* chan_shift, int64_t B, float* d_scores) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !d_white || !d_scores) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (B <= 0) return af_fail(ctx, AFRAME_EINVAL, "B must be positive");
  if (dtype != AFRAME_FP32 && dtype != AFRAME_BF16 && dtype != AFRAME_F16) return af_fail(ctx, AFRAME_EINVAL, "bad dtype");
  if (first < 0) return af_fail(ctx, AFRAME_EINVAL, "first must be non-negative");
  int64_t choff[AF_MAX_CH] = {0};
  for (int c = 0; c < ctx->cfg.n_channels; ++c) {
    const int64_t sh = chan_shift ? chan_shift[c] : 0;
    if (first + sh < 0 || first + sh + (B - 1) * ctx->cfg.stride + ctx->cfg.kernel_len > ld)
      return af_fail(ctx, AFRAME_ESHAPE, "windows reach outside the whitened stream (ld)");
    choff[c] = (int64_t)c * ld + first + sh;
  }
  return forward_common(ctx, w, d_white, (int)dtype, ctx->cfg.stride, choff, B, d_scores);
}

// ---- per-stage device timing --------------------------------------------------------------------------
static cudaEvent_t prof_event(aframe_ctx* ctx) {
  cudaEvent_t e = nullptr;
  if (!ctx->prof_pool.empty()) { e = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); return e; }
  if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return e;
}

void af_prof_begin(aframe_ctx* ctx, int kind) {
  if (!ctx->prof_on || ctx->prof_open[kind]) return;
  cudaEvent_t e = prof_event(ctx);
  if (!e) return;
  cudaEventRecord(e, ctx->stream);
  ctx->prof_open[kind] = e;
}

void af_prof_end(aframe_ctx* ctx, int kind, int launches) {
  if (!ctx->prof_on || !ctx->prof_open[kind]) return;
  cudaEvent_t e = prof_event(ctx);
  if (!e) return;
  cudaEventRecord(e, ctx->stream);
  ctx->prof_spans.push_back(ProfSpan{ctx->prof_open[kind], e, kind, launches});
  ctx->prof_open[kind] = nullptr;
}

static void prof_clear(aframe_ctx* ctx) {
  for (ProfSpan& s : ctx->prof_spans) { ctx->prof_pool.push_back(s.a); ctx->prof_pool.push_back(s.b); }
  ctx->prof_spans.clear();
  for (int k = 0; k < AFRAME_PROF_KINDS; ++k)
    if (ctx->prof_open[k]) { ctx->prof_pool.push_back(ctx->prof_open[k]); ctx->prof_open[k] = nullptr; }
}

AF_API aframe_status aframe_profile(aframe_ctx* ctx, int enable) {
  if (!ctx) return AFRAME_EINVAL;
  AF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  prof_clear(ctx);
  ctx->prof_on = enable != 0;
  return AFRAME_OK;
}

AF_API aframe_status aframe_profile_read(aframe_ctx* ctx, double* h_ms, int64_t* h_launches) {
  if (!ctx) return AFRAME_EINVAL;
  if (!h_ms || !h_launches) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  AF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  for (int k = 0; k < AFRAME_PROF_KINDS; ++k) { h_ms[k] = 0.0; h_launches[k] = 0; }
  for (const ProfSpan& s : ctx->prof_spans) {
    float ms = 0.f;
    AF_CUDA(ctx, cudaEventElapsedTime(&ms, s.a, s.b));
    h_ms[s.kind] += (double)ms;
    h_launches[s.kind] += s.launches;
  }
  return AFRAME_OK;
}

// ---- offline background analysis: whiten once, score every timeslide (configs[3]) ---------------------
static aframe_status score_timeslides_dev(aframe_ctx* ctx, const aframe_weights* w, const float* d_strain,
                                          int64_t n_samples, int64_t ld, int64_t first, int64_t n_windows,
                                          const int64_t* h_slide_shifts, int32_t n_slides, int64_t batch,
                                          float* d_scores) {
  const aframe_config& cfg = ctx->cfg;
  const int C = cfg.n_channels;
  if (n_windows <= 0 || n_slides <= 0 || batch <= 0) return af_fail(ctx, AFRAME_EINVAL, "n_windows, n_slides, batch must be positive");
  if (first < 0) return af_fail(ctx, AFRAME_EINVAL, "first must be non-negative");
  if (w->ctx != ctx) return af_fail(ctx, AFRAME_ESTATE, "weights belong to another context");
  // whitened stream in the network's input precision
  const aframe_precision wdt = cfg.precision == AFRAME_F16 ? AFRAME_F16 : AFRAME_FP32;
  const size_t esz = af_dt_bytes((int)wdt);
  const int64_t ld_w = (n_samples + 63) & ~(int64_t)63;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_white, esz * (size_t)C * ld_w);
  if (st != AFRAME_OK) return st;
  int64_t n_out = 0;
  st = aframe_whiten_rolling(ctx, d_strain, n_samples, ld, ctx->ws_white.ptr, ld_w, wdt, &n_out);
  if (st != AFRAME_OK) return st;
  int64_t sh_min = 0, sh_max = 0;
  for (int k = 0; k < n_slides; ++k) {
    if (h_slide_shifts[k] < sh_min) sh_min = h_slide_shifts[k];
    if (h_slide_shifts[k] > sh_max) sh_max = h_slide_shifts[k];
  }
  if (first + sh_min < 0 || first + sh_max + (n_windows - 1) * cfg.stride + cfg.kernel_len > n_out)
    return af_fail(ctx, AFRAME_ESHAPE, "timeslide windows reach outside the whitened segment");
  for (int k = 0; k < n_slides; ++k) {
    int64_t shifts[AF_MAX_CH];
    shifts[0] = 0;
    for (int c = 1; c < C; ++c) shifts[c] = h_slide_shifts[k];
    for (int64_t i0 = 0; i0 < n_windows; i0 += batch) {
      const int64_t nb = n_windows - i0 < batch ? n_windows - i0 : batch;
      st = aframe_forward_strided(ctx, w, ctx->ws_white.ptr, wdt, ld_w,
                                  first + i0 * cfg.stride, shifts, nb, d_scores + (int64_t)k * n_windows + i0);
      if (st != AFRAME_OK) return st;
    }
  }
  return AFRAME_OK;
}

AF_API aframe_status aframe_score_timeslides(aframe_ctx* ctx, const aframe_weights* w, const float* d_strain,
                                             int64_t n_samples, int64_t ld, int64_t first, int64_t n_windows,
                                             const int64_t* h_slide_shifts, int32_t n_slides, int64_t batch,
                                             float* d_scores) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !d_strain || !h_slide_shifts || !d_scores) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  return score_timeslides_dev(ctx, w, d_strain, n_samples, ld, first, n_windows, h_slide_shifts, n_slides, batch, d_scores);
}

AF_API aframe_status aframe_score_timeslides_host(aframe_ctx* ctx, const aframe_weights* w, const float* h_strain,
                                                  int64_t n_samples, int64_t ld, int64_t first, int64_t n_windows,
                                                  const int64_t* h_slide_shifts, int32_t n_slides, int64_t batch,
                                                  float* h_scores) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !h_strain || !h_slide_shifts || !h_scores) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (n_samples <= 0 || ld < n_samples) return af_fail(ctx, AFRAME_ESHAPE, "ld < n_samples");
  if (n_windows <= 0 || n_slides <= 0) return af_fail(ctx, AFRAME_EINVAL, "n_windows, n_slides must be positive");
  const int C = ctx->cfg.n_channels;
  const int64_t ld_d = (n_samples + 63) & ~(int64_t)63;
  const size_t strain_bytes = sizeof(float) * (size_t)C * ld_d;
  const size_t score_bytes = sizeof(float) * (size_t)n_slides * n_windows;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_stage, strain_bytes + score_bytes);
  if (st != AFRAME_OK) return st;
  float* d_strain = reinterpret_cast<float*>(ctx->ws_stage.ptr);
  float* d_scores = reinterpret_cast<float*>(reinterpret_cast<char*>(ctx->ws_stage.ptr) + strain_bytes);
  AF_CUDA(ctx, cudaMemcpy2DAsync(d_strain, sizeof(float) * ld_d, h_strain, sizeof(float) * ld, sizeof(float) * n_samples, C,
                                 cudaMemcpyHostToDevice, ctx->stream));
  st = score_timeslides_dev(ctx, w, d_strain, n_samples, ld_d, first, n_windows, h_slide_shifts, n_slides, batch, d_scores);
  if (st != AFRAME_OK) return st;
  AF_CUDA(ctx, cudaMemcpyAsync(h_scores, d_scores, score_bytes, cudaMemcpyDeviceToHost, ctx->stream));
  AF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  return AFRAME_OK;
}

AF_API aframe_status aframe_profile_layers(aframe_ctx* ctx, const aframe_weights* w, const float* d_windows, int64_t B,
                                           float* d_scores, float* h_ms, int32_t n_layers) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !d_windows || !d_scores || !h_ms) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (n_layers != (int32_t)w->layers.size()) return af_fail(ctx, AFRAME_ESHAPE, "n_layers does not match the layer table");
  if (ctx->cfg.precision != AFRAME_F16) return af_fail(ctx, AFRAME_EUNSUPPORTED, "per-layer timing is built for the tensor-core path");
  for (int i = 0; i < n_layers; ++i) h_ms[i] = 0.f;
  ctx->layer_ms = h_ms;
  aframe_status st = aframe_forward(ctx, w, d_windows, B, d_scores);
  ctx->layer_ms = nullptr;
  return st;
}
