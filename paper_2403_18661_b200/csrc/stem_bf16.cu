// Fused stem of the bf16 path: window assembly in place from the whitened stream,
// conv k7 s2 (C_in -> 64) + folded norm + ReLU + max-pool k3 s2 p1, output rounded once to bf16,
// channels-last [B][T_pool][C_out].  K = C_in*7 = 14 is not a tensor-core shape: fp32 FFMA on CUDA cores.
// The pre-pool tensor never leaves the SM.
#include "common.cuh"
#include "stem.h"

template <bool IN_BF16>
__device__ __forceinline__ float stem_ld(const void* p, int64_t i) {
  if (IN_BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[i]);
  return __ldg(reinterpret_cast<const float*>(p) + i);
}

// One CTA: one window, TP pooled positions, all C_OUT channels.  thread -> (co = tid % C_OUT, tq = tid / C_OUT).
template <bool IN_BF16, int KW, int CIN, int C_OUT, int TP>
__global__ void __launch_bounds__(256)
stem_pool_kernel(const void* __restrict__ in, int64_t sB, StemOff off, const float* __restrict__ w /*[KW][CIN][C_OUT]*/,
                 const float* __restrict__ bias, int T_in, int T_conv, int T_pool, __nv_bfloat16* __restrict__ out) {
  constexpr int PAD = KW / 2;
  constexpr int NX = 4 * TP + 2 * PAD + 1;          // input samples per channel needed by TP pooled outputs
  constexpr int TQ = 256 / C_OUT;
  __shared__ float xs[CIN][NX + 1];
  const int tid = threadIdx.x;
  const int64_t b = blockIdx.y;
  const int tp0 = blockIdx.x * TP;
  const int x0 = 4 * tp0 - 2 - PAD;                 // input index of xs[.][0]: conv pos 2*tp0-1 reads 2*(2tp0-1)-PAD..
  for (int i = tid; i < CIN * NX; i += 256) {
    const int c = i / NX, n = i - c * NX;
    const int t = x0 + n;
    xs[c][n] = (t >= 0 && t < T_in) ? stem_ld<IN_BF16>(in, b * sB + off.v[c] + t) : 0.f;
  }
  const int co = tid % C_OUT, tq = tid / C_OUT;
  float wr[KW][CIN];
#pragma unroll
  for (int d = 0; d < KW; ++d)
#pragma unroll
    for (int c = 0; c < CIN; ++c) wr[d][c] = w[(d * CIN + c) * C_OUT + co];
  const float bs = bias[co];
  __syncthreads();
  for (int tl = tq; tl < TP; tl += TQ) {
    const int tp = tp0 + tl;
    if (tp >= T_pool) break;
    // conv positions 2tp-1, 2tp, 2tp+1 read xs[c][4*tl + 2*e + d], e = 0..2, d = 0..KW-1
    float xr[CIN][KW + 4];
#pragma unroll
    for (int c = 0; c < CIN; ++c)
#pragma unroll
      for (int n = 0; n < KW + 4; ++n) xr[c][n] = xs[c][4 * tl + n];
    float best = 0.f;                                // post-ReLU values are >= 0, so 0 is the identity
#pragma unroll
    for (int e = 0; e < 3; ++e) {
      const int tc = 2 * tp + e - 1;
      float acc = bs;
#pragma unroll
      for (int d = 0; d < KW; ++d)
#pragma unroll
        for (int c = 0; c < CIN; ++c) acc = fmaf(wr[d][c], xr[c][2 * e + d], acc);
      if (tc >= 0 && tc < T_conv) best = fmaxf(best, acc);
    }
    out[((int64_t)b * T_pool + tp) * C_OUT + co] = __float2bfloat16_rn(best);
  }
}

aframe_status af_launch_stem_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                  int in_bf16, int64_t sB, const int64_t* choff, const float* d_w, const float* d_bias,
                                  int64_t B, __nv_bfloat16* d_out) {
  if (!(conv.k == 7 && conv.c_in == 2 && conv.c_out == 64 && conv.stride == 2 && conv.pad == 3 && conv.relu &&
        pool.k == 3 && pool.stride == 2 && pool.pad == 1))
    return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem: only conv(2->64,k7,s2,p3)+ReLU+maxpool(k3,s2,p1) is built");
  constexpr int TP = 64;
  StemOff off;
  for (int c = 0; c < AF_MAX_CH; ++c) off.v[c] = c < conv.c_in ? choff[c] : 0;
  dim3 grid((unsigned)((pool.t_out + TP - 1) / TP), (unsigned)B);
  if (in_bf16)
    stem_pool_kernel<true, 7, 2, 64, TP><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, conv.t_out,
                                                                        pool.t_out, d_out);
  else
    stem_pool_kernel<false, 7, 2, 64, TP><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, conv.t_out,
                                                                         pool.t_out, d_out);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
