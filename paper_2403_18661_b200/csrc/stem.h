#pragma once
#include "common.cuh"

struct StemOff { int64_t v[AF_MAX_CH]; };   // per-channel element offset of a window's first sample

aframe_status af_launch_stem_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                  int in_bf16, int64_t sB, const int64_t* choff, const float* d_w, const float* d_bias,
                                  int64_t B, __nv_bfloat16* d_out);
