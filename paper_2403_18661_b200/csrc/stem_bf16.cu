// Fused stem of the bf16 path: window assembly in place from the whitened stream,
// conv k7 s2 (C_in -> 64) + folded norm + ReLU + max-pool k3 s2 p1, output rounded once to fp16,
// channels-last [B][T_pool][C_out].  K = C_in*7 = 14 is not a tensor-core shape: fp32 FFMA on CUDA cores.
// The pre-pool tensor never leaves the SM.
#include "common.cuh"
#include "stem.h"

template <int IN_DT>
__device__ __forceinline__ float stem_ld(const void* p, int64_t i) { return af_ld_as_f32<IN_DT>(p, i); }

// One CTA: one window, TP pooled positions, all 64 channels.  lane <-> channel pair (2*lane, 2*lane+1), warp <-> a run
// of TP/8 consecutive pooled positions.  Each conv position is computed once per run (the pool's shared position is
// carried in a register), the input slides through registers as float4s, and a warp stores one 128-byte line per
// pooled position.
// GN (NEXT-2, true GroupNorm): the conv output is normalised with the window's own statistics before ReLU and pool,
// v = acc * sc + sh with sc = rstd_g gamma_c, sh = beta_c - mu_g rstd_g gamma_c (stats from stem_gn_stats_kernel).
template <int IN_DT, int TP, bool GN>
__global__ void __launch_bounds__(256)
stem_pool_kernel(const void* __restrict__ in, int64_t sB, StemOff off, const float* __restrict__ w /*[7][2][64]*/,
                 const float* __restrict__ bias, int T_in, int T_pool, af_act_t* __restrict__ out,
                 const float2* __restrict__ stats, const float* __restrict__ gamma, const float* __restrict__ beta, int G) {
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
    xs[c][n] = (t >= 0 && t < T_in) ? stem_ld<IN_DT>(in, b * sB + off.v[c] + t) : 0.f;
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
  float sc0 = 1.f, sc1 = 1.f, sh0 = 0.f, sh1 = 0.f;
  if (GN) {
    const int cg = C_OUT / G;
    const float2 st0 = stats[b * G + (2 * lane) / cg], st1 = stats[b * G + (2 * lane + 1) / cg];
    sc0 = st0.y * gamma[2 * lane]; sc1 = st1.y * gamma[2 * lane + 1];
    sh0 = beta[2 * lane] - st0.x * sc0; sh1 = beta[2 * lane + 1] - st1.x * sc1;
  }
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
    if (GN) { p0 = fmaf(p0, sc0, sh0); p1 = fmaf(p1, sc1, sh1); }
    p0 = fmaxf(p0, 0.f); p1 = fmaxf(p1, 0.f);
  }
  uint32_t* o = reinterpret_cast<uint32_t*>(out + ((int64_t)b * T_pool + tp0 + tl0) * C_OUT) + lane;
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
    if (GN) { a0 = fmaf(a0, sc0, sh0); a1 = fmaf(a1, sc1, sh1); c0 = fmaf(c0, sc0, sh0); c1 = fmaf(c1, sc1, sh1); }
    c0 = fmaxf(c0, 0.f); c1 = fmaxf(c1, 0.f);
    const float m0 = fmaxf(fmaxf(p0, a0), c0), m1 = fmaxf(fmaxf(p1, a1), c1);   // ReLU folded: p, c >= 0
    if (tp0 + tl0 + i < T_pool) o[(int64_t)i * (C_OUT / 2)] = af_act_pack2(m0, m1);
    p0 = c0; p1 = c1;
#pragma unroll
    for (int c = 0; c < CIN; ++c)
#pragma unroll
      for (int k = 0; k < 8; ++k) r[c][k] = r[c][k + 4];
  }
}

// NEXT-2: per (window, group) mean and 1/sqrt(var + eps) of the stem conv output (biased variance over the group's
// channels and all T_conv positions), computed without storing the conv output.  One CTA per window; lane <->
// channel pair, each warp walks pairs of conv positions (2u, 2u+1), which read x[4u-3 .. 4u+5].
template <int IN_DT>
__global__ void __launch_bounds__(256)
stem_gn_stats_kernel(const void* __restrict__ in, int64_t sB, StemOff off, const float* __restrict__ w /*[7][2][64]*/,
                     const float* __restrict__ bias, int T_in, int G, float eps, float2* __restrict__ stats) {
  constexpr int KW = 7, CIN = 2, C_OUT = 64;
  extern __shared__ __align__(16) float xs_dyn[];     // [CIN][T_in + 8], xs[c][n] = x[c][n - 4]
  __shared__ double red_s[8][32], red_q[8][32];
  const int NX = T_in + 8;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t b = blockIdx.x;
  for (int i = tid; i < CIN * NX; i += 256) {
    const int c = i / NX, n = i - c * NX;
    const int t = n - 4;
    xs_dyn[i] = (t >= 0 && t < T_in) ? stem_ld<IN_DT>(in, b * sB + off.v[c] + t) : 0.f;
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
  double S = 0.0, Q = 0.0;                             // both channels of the pair are in the same group (C_OUT / G even)
  const int n_pairs = T_in / 4;
  for (int u0 = warp * 32; u0 < n_pairs; u0 += 8 * 32) {
    float s = 0.f, q = 0.f;                            // fp32 over a run of 32 position pairs, double across runs
    const int u1 = u0 + 32 < n_pairs ? u0 + 32 : n_pairs;
    for (int u = u0; u < u1; ++u) {
      float r[CIN][12];                                // x[4u-4 .. 4u+8)
#pragma unroll
      for (int c = 0; c < CIN; ++c)
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const float4 v = *reinterpret_cast<const float4*>(&xs_dyn[c * NX + 4 * u + 4 * k]);
          r[c][4 * k] = v.x; r[c][4 * k + 1] = v.y; r[c][4 * k + 2] = v.z; r[c][4 * k + 3] = v.w;
        }
      float a0 = bs.x, a1 = bs.y, c0 = bs.x, c1 = bs.y;
#pragma unroll
      for (int c = 0; c < CIN; ++c)
#pragma unroll
        for (int d = 0; d < KW; ++d) {
          a0 = fmaf(w0[d][c], r[c][1 + d], a0); a1 = fmaf(w1[d][c], r[c][1 + d], a1);
          c0 = fmaf(w0[d][c], r[c][3 + d], c0); c1 = fmaf(w1[d][c], r[c][3 + d], c1);
        }
      s += (a0 + a1) + (c0 + c1);
      q = fmaf(a0, a0, q); q = fmaf(a1, a1, q); q = fmaf(c0, c0, q); q = fmaf(c1, c1, q);
    }
    S += (double)s; Q += (double)q;
  }
  red_s[warp][lane] = S; red_q[warp][lane] = Q;
  __syncthreads();
  if (tid < G) {
    const int lg = (C_OUT / G) / 2;                    // lanes per group
    double ts = 0.0, tq = 0.0;
    for (int wv = 0; wv < 8; ++wv)
      for (int l = tid * lg; l < (tid + 1) * lg; ++l) { ts += red_s[wv][l]; tq += red_q[wv][l]; }
    const double n = (double)(T_in / 2) * (C_OUT / G), mu = ts / n;
    const double var = tq / n - mu * mu;
    stats[b * G + tid] = make_float2((float)mu, (float)(1.0 / sqrt((var > 0.0 ? var : 0.0) + (double)eps)));
  }
}

// Shared stem (overlapping windows): rows 0, 1 and T_pool - 1 of every window are the only pooled rows that see the
// window's own zero padding; everything else equals the stem of the whole stream (af_launch_stem_stream_bf16).  One warp
// per window, lane <-> channel pair; the FMA order is the one of stem_pool_kernel, so the values are bit-identical to
// what the per-window kernel stores.  edge: [nb][3][64] fp16 (rows 0, 1, T_pool - 1).
template <int IN_DT>
__global__ void __launch_bounds__(128)
stem_edge_kernel(const void* __restrict__ in, int64_t sB, StemOff off, const float* __restrict__ w /*[7][2][64]*/,
                 const float* __restrict__ bias, int T_in, int T_pool, int64_t nb, af_act_t* __restrict__ edge) {
  constexpr int KW = 7, CIN = 2, C_OUT = 64;
  const int lane = threadIdx.x & 31;
  const int64_t b = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (b >= nb) return;
  float w0[KW][CIN], w1[KW][CIN];
#pragma unroll
  for (int d = 0; d < KW; ++d)
#pragma unroll
    for (int c = 0; c < CIN; ++c) {
      const float2 ww = *reinterpret_cast<const float2*>(w + (d * CIN + c) * C_OUT + 2 * lane);
      w0[d][c] = ww.x; w1[d][c] = ww.y;
    }
  const float2 bs = *reinterpret_cast<const float2*>(bias + 2 * lane);
  const int T_conv = T_in / 2;
#pragma unroll 1
  for (int k = 0; k < 3; ++k) {
    const int u = k < 2 ? k : T_pool - 1;
    float m0 = 0.f, m1 = 0.f;                          // ReLU folded into the max
#pragma unroll 1
    for (int t = 2 * u - 1; t <= 2 * u + 1; ++t) {
      if (t < 0 || t >= T_conv) continue;              // pool padding never wins
      float a0 = bs.x, a1 = bs.y;
#pragma unroll
      for (int c = 0; c < CIN; ++c)
#pragma unroll
        for (int d = 0; d < KW; ++d) {
          const int x = 2 * t - 3 + d;
          const float xv = (x >= 0 && x < T_in) ? stem_ld<IN_DT>(in, b * sB + off.v[c] + x) : 0.f;
          a0 = fmaf(w0[d][c], xv, a0); a1 = fmaf(w1[d][c], xv, a1);
        }
      m0 = fmaxf(m0, a0); m1 = fmaxf(m1, a1);
    }
    reinterpret_cast<uint32_t*>(edge + (b * 3 + k) * C_OUT)[lane] = af_act_pack2(m0, m1);
  }
}

// Shared stem: the windows of one launch are K-sample views at a spacing of win_stride samples (a multiple of 4) into
// one whitened stream, so their pooled stem outputs are views at a spacing of win_stride / 4 rows into the stem of the
// whole stream, except for the three rows above.  d_stream: [(nb - 1) * win_stride / 4 + T_pool][64] fp16.
aframe_status af_launch_stem_stream_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                         int in_dt, int64_t win_stride, const int64_t* choff, const float* d_w,
                                         const float* d_bias, int64_t nb, af_act_t* d_stream, af_act_t* d_edge) {
  constexpr int TP = 128;
  StemOff off;
  for (int c = 0; c < AF_MAX_CH; ++c) off.v[c] = c < conv.c_in ? choff[c] : 0;
  const int64_t T_in = (nb - 1) * win_stride + conv.t_in;
  if (T_in > (1ll << 30)) return af_fail(ctx, AFRAME_ESHAPE, "shared stem: stream longer than 2^30 samples");
  const int T_pool = (int)(T_in / 4);
  dim3 grid((unsigned)((T_pool + TP - 1) / TP), 1);
#define AF_STEM_STREAM(DT)                                                                                              \
  do {                                                                                                                  \
    stem_pool_kernel<DT, TP, false><<<grid, 256, 0, ctx->stream>>>(d_in, 0, off, d_w, d_bias, (int)T_in, T_pool, d_stream, \
                                                                   nullptr, nullptr, nullptr, 1);                        \
    AF_LAUNCH_CHECK(ctx);                                                                                               \
    stem_edge_kernel<DT><<<(unsigned)((nb + 3) / 4), 128, 0, ctx->stream>>>(d_in, win_stride, off, d_w, d_bias, conv.t_in, \
                                                                            pool.t_out, nb, d_edge);                     \
  } while (0)
  if (in_dt == AF_DT_BF16) AF_STEM_STREAM(AF_DT_BF16);
  else if (in_dt == AF_DT_F16) AF_STEM_STREAM(AF_DT_F16);
  else AF_STEM_STREAM(AF_DT_F32);
#undef AF_STEM_STREAM
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

aframe_status af_launch_stem_bf16(aframe_ctx* ctx, const LayerDesc& conv, const LayerDesc& pool, const void* d_in,
                                  int in_dt, int64_t sB, const int64_t* choff, const float* d_w, const float* d_bias,
                                  int64_t B, af_act_t* d_out, const StemGn* gn) {
  if (!(conv.k == 7 && conv.c_in == 2 && conv.c_out == 64 && conv.stride == 2 && conv.pad == 3 && conv.relu &&
        pool.k == 3 && pool.stride == 2 && pool.pad == 1))
    return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem: only conv(2->64,k7,s2,p3)+ReLU+maxpool(k3,s2,p1) is built");
  constexpr int TP = 128;   // pooled positions per CTA (measured on B200, 4096 windows: 64 -> 355 us, 128 -> 321 us, 256 -> 353 us)
  if (conv.t_out != 2 * pool.t_out || conv.t_in != 2 * conv.t_out)
    return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem: input length must be a multiple of 4");
  StemOff off;
  for (int c = 0; c < AF_MAX_CH; ++c) off.v[c] = c < conv.c_in ? choff[c] : 0;
  dim3 grid((unsigned)((pool.t_out + TP - 1) / TP), (unsigned)B);
  if (gn) {
    const size_t smem = sizeof(float) * 2 * (size_t)(conv.t_in + 8);
    if (gn->G < 1 || gn->G > 32 || 64 % gn->G || (64 / gn->G) % 2 || smem > 48 * 1024)
      return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 stem with true GroupNorm: needs an even number of channels per group and kernel_len <= 6136");
#define AF_STEM_GN(DT)                                                                                                  \
  do {                                                                                                                  \
    stem_gn_stats_kernel<DT><<<(unsigned)B, 256, smem, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, gn->G, gn->eps, gn->stats); \
    stem_pool_kernel<DT, TP, true><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out, \
                                                                  gn->stats, gn->gamma, gn->beta, gn->G);                \
  } while (0)
    if (in_dt == AF_DT_BF16) AF_STEM_GN(AF_DT_BF16);
    else if (in_dt == AF_DT_F16) AF_STEM_GN(AF_DT_F16);
    else AF_STEM_GN(AF_DT_F32);
#undef AF_STEM_GN
    ctx->launches++;
  } else if (in_dt == AF_DT_BF16)
    stem_pool_kernel<AF_DT_BF16, TP, false><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out,
                                                                           nullptr, nullptr, nullptr, 1);
  else if (in_dt == AF_DT_F16)
    stem_pool_kernel<AF_DT_F16, TP, false><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out,
                                                                          nullptr, nullptr, nullptr, 1);
  else
    stem_pool_kernel<AF_DT_F32, TP, false><<<grid, 256, 0, ctx->stream>>>(d_in, sB, off, d_w, d_bias, conv.t_in, pool.t_out, d_out,
                                                                          nullptr, nullptr, nullptr, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
