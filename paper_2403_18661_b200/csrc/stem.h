#pragma once
#include "common.cuh"

struct StemOff { int64_t v[AF_MAX_CH]; };   // per-channel element offset of a window's first sample

// true GroupNorm of the stem (NEXT-2): scratch for the per-window statistics and the affine parameters
struct StemGn { float2* stats; const float* gamma; const float* beta; int G; float eps; };

aframe_status af_launch_stem_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                  int in_dt, int64_t sB, const int64_t* choff, const float* d_w, const float* d_bias,
                                  int64_t B, af_act_t* d_out, const StemGn* gn = nullptr);

// shared stem of overlapping in-place windows (see stem_bf16.cu): stem of the whole stream + per-window edge rows
aframe_status af_launch_stem_stream_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                         int in_dt, int64_t win_stride, const int64_t* choff, const float* d_w,
                                         const float* d_bias, int64_t nb, af_act_t* d_stream, af_act_t* d_edge);

// true GroupNorm after a tensor-core conv (NEXT-2): statistics per (window, group), then normalise + affine (+ residual)
// (ReLU) in place on the fp16 tensor z [nb][T][C]; stats is scratch for nb * G float2.  partials != null: the conv epilogue
// already emitted per-slab partial sums of its fp32 accumulators (TcConvParams::gn_part); they are only combined here.
aframe_status af_launch_gn_bf16(aframe_ctx* ctx, af_act_t* z, const af_act_t* res, int T, int C, int G, float eps,
                                const float* gamma, const float* beta, int relu, int64_t nb, float2* stats,
                                const float2* partials = nullptr, int gn_unit = 0);
