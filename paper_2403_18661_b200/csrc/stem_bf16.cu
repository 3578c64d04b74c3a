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

// One CTA: one window, TP pooled positions, all 64 channels.  lane <-> channel pair (2*lane, 2*lane+1), warp <-> a run
// of TP/8 consecutive pooled positions.  Each conv position is computed once per run (the pool's shared position is
// carried in a register), the input slides through registers as float4s, and a warp stores one 128-byte line per
// pooled position.
template <bool IN_BF16, int TP>
__global__ void __launch_bounds__(256)
stem_pool_kernel(const void* __restrict__ in, int64_t sB, StemOff off, const float* __restrict__ w /*[7][2][64]*/,
                 const float* __restrict__ bias, int T_in, int T_pool, __nv_bfloat16* __restrict__ out) {
  constexpr int KW = 7, CIN = 2, C_OUT = 64;
  constexpr int RUN = TP / 8;
  constexpr int NX = 4 * TP + 16;                    // samples x[4 tp0 - 8 .. 4 tp0 + 4 TP + 8) per channel
  __shared__ __align__(16) float xs[CIN][NX];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t b = blockIdx.y;
  const int tp0 = blockIdx.x * TP;
  const int x0 = 4 * tp0 - 8;
  for (int i = tid; i < CIN * NX; i += 256) {
    const int c = i / NX, n = i - c * NX;
    const int t = x0 + n;
    xs[c][n] = (t >= 0 && t < T_in) ? stem_ld<IN_BF16>(in, b * sB + off.v[c] + t) : 0.f;
  }
  float w0[KW][CIN], w1[KW][CIN];
#pragma unroll
  for (int d = 0; d < KW; ++d)
#pragma unroll
    for (int c = 0; c < CIN; ++c) {
      const float2 ww = *reinterpret_cast<const float2*>(w + (d * CIN + c) * C_OUT + 2 * lane);
      w0[d][c] = ww.x; w1[d][c] = ww.y;
    }
  const float2 bs = *reinterpret_cast<const float2*>(bias + 2 * lane);
  __syncthreads();

  const int tl0 = warp * RUN;                        // first pooled position (local) of this warp's run
  // r[c][0..11] = x[c][4 tp - 4 .. 4 tp + 8)  (xs index 4 tl + 4 + i)
  float r[CIN][12];
#pragma unroll
  for (int c = 0; c < CIN; ++c) {
    const float4 a = *reinterpret_cast<const float4*>(&xs[c][4 * tl0 + 4]);
    const float4 bq = *reinterpret_cast<const float4*>(&xs[c][4 * tl0 + 8]);
    r[c][0] = a.x; r[c][1] = a.y; r[c][2] = a.z; r[c][3] = a.w;
    r[c][4] = bq.x; r[c][5] = bq.y; r[c][6] = bq.z; r[c][7] = bq.w;
  }
  // conv position 2 tp - 1 of the run's first tp reads x[4 tp - 5 .. 4 tp + 1]
  float p0 = 0.f, p1 = 0.f;
  if (tp0 + tl0 > 0) {
    p0 = bs.x; p1 = bs.y;
#pragma unroll
    for (int c = 0; c < CIN; ++c) {
      const float xm = xs[c][4 * tl0 + 3];           // x[4 tp - 5]
#pragma unroll
      for (int d = 0; d < KW; ++d) {
        const float xv = d == 0 ? xm : r[c][d - 1];
        p0 = fmaf(w0[d][c], xv, p0); p1 = fmaf(w1[d][c], xv, p1);
      }
    }
    p0 = fmaxf(p0, 0.f); p1 = fmaxf(p1, 0.f);
  }
  __nv_bfloat162* o = reinterpret_cast<__nv_bfloat162*>(out + ((int64_t)b * T_pool + tp0 + tl0) * C_OUT) + lane;
#pragma unroll
  for (int i = 0; i < RUN; ++i) {
#pragma unroll
    for (int c = 0; c < CIN; ++c) {
      const float4 nq = *reinterpret_cast<const float4*>(&xs[c][4 * (tl0 + i) + 12]);
      r[c][8] = nq.x; r[c][9] = nq.y; r[c][10] = nq.z; r[c][11] = nq.w;
    }
    float a0 = bs.x, a1 = bs.y, c0 = bs.x, c1 = bs.y;   // conv positions 2 tp (x[4tp-3..]) and 2 tp + 1 (x[4tp-1..])
#pragma unroll
    for (int c = 0; c < CIN; ++c)
#pragma unroll
      for (int d = 0; d < KW; ++d) {
        a0 = fmaf(w0[d][c], r[c][1 + d], a0); a1 = fmaf(w1[d][c], r[c][1 + d], a1);
        c0 = fmaf(w0[d][c], r[c][3 + d], c0); c1 = fmaf(w1[d][c], r[c][3 + d], c1);
      }
    c0 = fmaxf(c0, 0.f); c1 = fmaxf(c1, 0.f);
    const float m0 = fmaxf(fmaxf(p0, a0), c0), m1 = fmaxf(fmaxf(p1, a1), c1);   // ReLU folded: p, c >= 0
    if (tp0 + tl0 + i < T_pool) o[(int64_t)i * (C_OUT / 2)] = __floats2bfloat162_rn(m0, m1);
    p0 = c0; p1 = c1;
#pragma unroll
    for (int c = 0; c < CIN; ++c)
#pragma unroll
      for (int k = 0; k < 8; ++k) r[c][k] = r[c][k + 4];
  }
}

aframe_status af_launch_stem_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                  int in_bf16, int64_t sB, const int64_t* choff, const float* d_w, const float* d_bias,
                                  int64_t B, __nv_bfloat16* d_out) {
  if (!(conv.k == 7 && conv.c_in == 2 && conv.c_out == 64 && conv.stride == 2 && conv.pad == 3 && conv.relu &&
        pool.k == 3 && pool.stride == 2 && pool.pad == 1))
    return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem: only conv(2->64,k7,s2,p3)+ReLU+maxpool(k3,s2,p1) is built");
  constexpr int TP = 64;
  if (conv.t_out != 2 * pool.t_out || conv.t_in != 2 * conv.t_out)
    return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem: input length must be a multiple of 4");
  StemOff off;
  for (int c = 0; c < AF_MAX_CH; ++c) off.v[c] = c < conv.c_in ? choff[c] : 0;
  dim3 grid((unsigned)((pool.t_out + TP - 1) / TP), (unsigned)B);
  if (in_bf16)
    stem_pool_kernel<true, TP><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out);
  else
    stem_pool_kernel<false, TP><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
