// NEXT-2, true GroupNorm on the tensor-core path ("GroupNorm ... whose statistics are computed per sample at inference").
// The tensor-core conv stores its plain output z (no bias, no ReLU, no residual) as fp16 [B][T][C]; these two kernels
// then compute, per (window, group), the mean and biased variance over the group's channels and all T positions and
// apply y = (z - mu) rstd gamma_c + beta_c (+ residual) (ReLU) in place.  Both are pure HBM streams: 16-byte accesses,
// one CTA per window for the statistics, one thread per 8 channels for the apply.
#include "common.cuh"
#include "stem.h"

__device__ __forceinline__ void gn_unpack8(const uint4 v, float* f) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float2 t = af_act_unpack2(w[j]);
    f[2 * j] = t.x; f[2 * j + 1] = t.y;
  }
}

// Fast path: C/8 divides 256 (so a thread always sees the same 8 channels) and a group is a whole number of octets.
__global__ void __launch_bounds__(256)
gn_stats_bf16_kernel(const af_act_t* __restrict__ z, int T, int C, int G, float eps, float2* __restrict__ stats) {
  __shared__ double rs[256], rq[256];
  const int64_t b = blockIdx.x;
  const int opr = C / 8;                               // octets per row
  const int n_oct = T * opr;
  const uint4* zb = reinterpret_cast<const uint4*>(z + b * (int64_t)T * C);
  double S = 0.0, Q = 0.0;
#pragma unroll 4
  for (int i = threadIdx.x; i < n_oct; i += 256) {
    float f[8];
    gn_unpack8(zb[i], f);
    float s = 0.f, q = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) { s += f[j]; q = fmaf(f[j], f[j], q); }
    S += (double)s; Q += (double)q;
  }
  rs[threadIdx.x] = S; rq[threadIdx.x] = Q;
  __syncthreads();
  if ((int)threadIdx.x < G) {
    const int opg = (C / G) / 8;                       // octets per group
    double ts = 0.0, tq = 0.0;
    for (int t = 0; t < 256; ++t)
      if ((t % opr) / opg == (int)threadIdx.x) { ts += rs[t]; tq += rq[t]; }
    const double n = (double)T * (C / G), mu = ts / n;
    const double var = tq / n - mu * mu;
    stats[b * G + threadIdx.x] = make_float2((float)mu, (float)(1.0 / sqrt((var > 0.0 ? var : 0.0) + (double)eps)));
  }
}

// General shapes: one CTA per (window, group), scalar loads.
__global__ void __launch_bounds__(256)
gn_stats_bf16_generic_kernel(const af_act_t* __restrict__ z, int T, int C, int G, float eps, float2* __restrict__ stats) {
  __shared__ double rs[8], rq[8];
  const int64_t b = blockIdx.x;
  const int g = blockIdx.y;
  const int cg = C / G;
  const af_act_t* zb = z + b * (int64_t)T * C + g * cg;
  double s = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < T * cg; i += blockDim.x) {
    const double v = (double)__half2float(zb[(int64_t)(i / cg) * C + (i % cg)]);
    s += v; q += v * v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); q += __shfl_xor_sync(0xffffffffu, q, o); }
  if ((threadIdx.x & 31) == 0) { rs[threadIdx.x >> 5] = s; rq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double ts = 0.0, tq = 0.0;
    for (int i = 0; i < 8; ++i) { ts += rs[i]; tq += rq[i]; }
    const double n = (double)T * cg, mu = ts / n;
    const double var = tq / n - mu * mu;
    stats[b * G + g] = make_float2((float)mu, (float)(1.0 / sqrt((var > 0.0 ? var : 0.0) + (double)eps)));
  }
}

// Statistics from the partial sums the conv epilogue emitted from its fp32 accumulators (conv_tc_kernel, gn_part):
// per (window, group) a fixed-order double sum over the T/32 slabs and the group's units.
__global__ void gn_finalize_kernel(const float2* __restrict__ part, int n_slabs, int n_units, int G, double n_elems, float eps,
                                   float2* __restrict__ stats) {
  const int64_t b = blockIdx.x;
  const int g = threadIdx.x;
  if (g >= G) return;
  const int upg = n_units / G;                         // units per group
  const float2* pb = part + b * (int64_t)n_slabs * n_units + g * upg;
  double ts = 0.0, tq = 0.0;
  for (int s = 0; s < n_slabs; ++s)
    for (int u = 0; u < upg; ++u) { const float2 v = pb[(int64_t)s * n_units + u]; ts += (double)v.x; tq += (double)v.y; }
  const double mu = ts / n_elems, var = tq / n_elems - mu * mu;
  stats[b * G + g] = make_float2((float)mu, (float)(1.0 / sqrt((var > 0.0 ? var : 0.0) + (double)eps)));
}

// Fast path (256 % (C/8) == 0): a CTA takes GN_ITER * 256 consecutive 8-channel octets of ONE window, so a thread always
// sees the same 8 channels: its 8 (scale, shift) pairs -- scale = rstd_g gamma_c, shift = beta_c - mu_g scale -- are set
// up once and every octet costs one 16-byte load (two with a residual), 8 FMAs and one 16-byte store.
constexpr int GN_ITER = 4;
template <bool RES>
__global__ void __launch_bounds__(256)
gn_apply_bf16_kernel(af_act_t* __restrict__ z, const float2* __restrict__ stats, const float* __restrict__ gamma,
                     const float* __restrict__ beta, const af_act_t* __restrict__ res, int n_oct_win /* T * C/8 */,
                     int segs /* CTAs per window */, int C, int G, int relu) {
  const int b = blockIdx.x / segs, seg = blockIdx.x - b * segs;
  const int opr = C / 8, cg = C / G;
  const int c0 = (threadIdx.x % opr) * 8;
  float sc[8], sh[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const float2 st = stats[(int64_t)b * G + (c0 + j) / cg];
    sc[j] = st.y * gamma[c0 + j];
    sh[j] = fmaf(-st.x, sc[j], beta[c0 + j]);
  }
  uint4* zb = reinterpret_cast<uint4*>(z) + (int64_t)b * n_oct_win;
  const uint4* rb = RES ? reinterpret_cast<const uint4*>(res) + (int64_t)b * n_oct_win : nullptr;
  const int i0 = seg * (GN_ITER * 256) + threadIdx.x;
  uint4 zv[GN_ITER], rv[GN_ITER];
#pragma unroll
  for (int k = 0; k < GN_ITER; ++k) {
    const int i = i0 + k * 256;
    if (i < n_oct_win) { zv[k] = zb[i]; if (RES) rv[k] = rb[i]; }
  }
#pragma unroll
  for (int k = 0; k < GN_ITER; ++k) {
    const int i = i0 + k * 256;
    if (i >= n_oct_win) continue;
    float f[8], r[8];
    gn_unpack8(zv[k], f);
    if (RES) gn_unpack8(rv[k], r);
    uint4 o;
    uint32_t* oh = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
    for (int j = 0; j < 8; j += 2) {
      float y0 = fmaf(f[j], sc[j], sh[j]), y1 = fmaf(f[j + 1], sc[j + 1], sh[j + 1]);
      if (RES) { y0 += r[j]; y1 += r[j + 1]; }
      if (relu) { y0 = fmaxf(y0, 0.f); y1 = fmaxf(y1, 0.f); }
      oh[j / 2] = af_act_pack2(y0, y1);
    }
    zb[i] = o;
  }
}

// General shapes (C/8 does not divide 256): one thread per octet.
template <bool RES>
__global__ void __launch_bounds__(256)
gn_apply_bf16_generic_kernel(af_act_t* __restrict__ z, const float2* __restrict__ stats, const float* __restrict__ gamma,
                             const float* __restrict__ beta, const af_act_t* __restrict__ res, int64_t n_oct, int T, int C,
                             int G, int relu) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_oct) return;
  const int opr = C / 8;
  const int c0 = (int)(i % opr) * 8;
  const int64_t b = i / ((int64_t)T * opr);
  const int cg = C / G;
  uint4* zp = reinterpret_cast<uint4*>(z) + i;
  float f[8], r[8];
  gn_unpack8(*zp, f);
  if (RES) gn_unpack8(reinterpret_cast<const uint4*>(res)[i], r);
  uint4 o;
  uint32_t* oh = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
  for (int j = 0; j < 8; j += 2) {
    float v[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const float2 st = stats[b * G + (c0 + j + k) / cg];
      const float scale = st.y * gamma[c0 + j + k];
      float y = fmaf(f[j + k], scale, fmaf(-st.x, scale, beta[c0 + j + k]));
      if (RES) y += r[j + k];
      if (relu) y = fmaxf(y, 0.f);
      v[k] = y;
    }
    oh[j / 2] = af_act_pack2(v[0], v[1]);
  }
  *zp = o;
}

aframe_status af_launch_gn_bf16(aframe_ctx* ctx, af_act_t* z, const af_act_t* res, int T, int C, int G, float eps,
                                const float* gamma, const float* beta, int relu, int64_t nb, float2* stats,
                                const float2* partials, int gn_unit) {
  if (C % 8 || G < 1 || C % G) return af_fail(ctx, AFRAME_EUNSUPPORTED, "bf16 GroupNorm: channels must be a multiple of 8 and of n_groups");
  const int opr = C / 8, cg = C / G;
  if (partials)
    gn_finalize_kernel<<<(unsigned)nb, (unsigned)((G + 31) / 32 * 32), 0, ctx->stream>>>(partials, T / 32, C / gn_unit, G, (double)T * cg,
                                                                                   eps, stats);
  else if (256 % opr == 0 && cg % 8 == 0 && G <= 256)
    gn_stats_bf16_kernel<<<(unsigned)nb, 256, 0, ctx->stream>>>(z, T, C, G, eps, stats);
  else
    gn_stats_bf16_generic_kernel<<<dim3((unsigned)nb, (unsigned)G), 256, 0, ctx->stream>>>(z, T, C, G, eps, stats);
  AF_LAUNCH_CHECK(ctx);
  const int64_t n_oct = nb * T * opr;
#define AF_GN_APPLY(RES_)                                                                                                \
  do {                                                                                                                  \
    if (256 % opr == 0 && (int64_t)T * opr < (1 << 30)) {                                                               \
      const int n_win = T * opr, segs = (n_win + GN_ITER * 256 - 1) / (GN_ITER * 256);                                  \
      gn_apply_bf16_kernel<RES_><<<(unsigned)(nb * segs), 256, 0, ctx->stream>>>(z, stats, gamma, beta, res, n_win, \
                                                                                       segs, C, G, relu);               \
    } else {                                                                                                            \
      gn_apply_bf16_generic_kernel<RES_><<<(unsigned)((n_oct + 255) / 256), 256, 0, ctx->stream>>>(               \
          z, stats, gamma, beta, res, n_oct, T, C, G, relu);                                                            \
    }                                                                                                                   \
  } while (0)
  if (res) AF_GN_APPLY(true); else AF_GN_APPLY(false);
#undef AF_GN_APPLY
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
