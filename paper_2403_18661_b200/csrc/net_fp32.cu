// fp32 CUDA-core network path (O-5): generic conv1d as a tiled implicit GEMM with fused folded-norm
// bias, residual add and ReLU; max-pool; global-average-pool + linear head.  Used for BASELINE.json
// configs[0] (whose channel counts are too small for UMMA tiles) and as the fp32 arm of configs[1].
// Activations are channels-last [B][T][C] fp32.
#include "common.cuh"
#include "net_plan.h"

struct ConvArgs {
  const void* in;
  int64_t in_sB, in_sT, in_sC;
  int64_t choff[AF_MAX_CH];
  int use_choff;
  const float* w;      // [k][c_in][c_out]
  const float* bias;   // [c_out]
  const float* res;    // [B][T_out][C_out] or null
  float* out;          // [B][T_out][C_out]
  int64_t rows;        // B * T_out
  int T_in, T_out, C_in, C_out, k, stride, pad, relu;
};

template <int IN_DT>
__device__ __forceinline__ float ld_in(const void* p, int64_t i) { return af_ld_as_f32<IN_DT>(p, i); }

template <int IN_DT>
__global__ void __launch_bounds__(256) conv_fp32_kernel(const ConvArgs a) {
  constexpr int BM = 64, BN = 64, BK = 16;
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN];
  const int tid = threadIdx.x;
  const int ty = tid >> 4, tx = tid & 15;
  const int64_t m0 = (int64_t)blockIdx.x * BM;
  const int n0 = blockIdx.y * BN;
  const int Ktot = a.k * a.C_in;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

  for (int k0 = 0; k0 < Ktot; k0 += BK) {
#pragma unroll
    for (int it = 0; it < (BM * BK) / 256; ++it) {
      const int idx = tid + it * 256;
      const int r = idx / BK, kk = idx % BK;
      const int64_t row = m0 + r;
      const int K = k0 + kk;
      float v = 0.f;
      if (row < a.rows && K < Ktot) {
        const int64_t b = row / a.T_out;
        const int t = (int)(row - b * a.T_out);
        const int d = K / a.C_in, ci = K - d * a.C_in;
        const int t_in = t * a.stride + d - a.pad;
        if (t_in >= 0 && t_in < a.T_in) {
          const int64_t off = b * a.in_sB + (int64_t)t_in * a.in_sT + (a.use_choff ? a.choff[ci] : (int64_t)ci * a.in_sC);
          v = ld_in<IN_DT>(a.in, off);
        }
      }
      As[kk][r] = v;
    }
#pragma unroll
    for (int it = 0; it < (BK * BN) / 256; ++it) {
      const int idx = tid + it * 256;
      const int kk = idx / BN, cc = idx % BN;
      const int K = k0 + kk, n = n0 + cc;
      Bs[kk][cc] = (K < Ktot && n < a.C_out) ? a.w[(int64_t)K * a.C_out + n] : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float av[4], bv[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) av[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) bv[j] = Bs[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t row = m0 + ty * 4 + i;
    if (row >= a.rows) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= a.C_out) continue;
      float v = acc[i][j] + a.bias[n];
      if (a.res) v += a.res[row * a.C_out + n];
      if (a.relu) v = fmaxf(v, 0.f);
      a.out[row * a.C_out + n] = v;
    }
  }
}

// NEXT-2, true GroupNorm: per (window, group) mean and biased variance over the group's channels and all time
// steps of the conv output z [B][T][C]; then y = (z - mu) rstd gamma_c + beta_c (+ residual) (ReLU), in place.
__global__ void __launch_bounds__(256) gn_stats_kernel(const float* __restrict__ z, int T, int C, int G, float eps,
                                                       float2* __restrict__ stats /*[B][G] (mu, rstd)*/) {
  __shared__ double rs[8], rq[8];
  const int64_t b = blockIdx.x;
  const int g = blockIdx.y;
  const int cg = C / G;
  const float* zb = z + b * (int64_t)T * C + g * cg;
  double s = 0.0, q = 0.0;
  for (int i = threadIdx.x; i < T * cg; i += blockDim.x) {
    const double v = (double)zb[(int64_t)(i / cg) * C + (i % cg)];
    s += v; q += v * v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); q += __shfl_xor_sync(0xffffffffu, q, o); }
  if ((threadIdx.x & 31) == 0) { rs[threadIdx.x >> 5] = s; rq[threadIdx.x >> 5] = q; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double ts = 0.0, tq = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { ts += rs[i]; tq += rq[i]; }
    const double n = (double)T * cg, mu = ts / n;
    const double var = tq / n - mu * mu;
    stats[b * G + g] = make_float2((float)mu, (float)(1.0 / sqrt((var > 0.0 ? var : 0.0) + (double)eps)));
  }
}

__global__ void gn_apply_kernel(float* __restrict__ z, const float2* __restrict__ stats, const float* __restrict__ gamma,
                                const float* __restrict__ beta, const float* __restrict__ res, int64_t total, int T, int C,
                                int G, int relu) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total) return;
  const int c = (int)(i % C);
  const int64_t b = i / ((int64_t)T * C);
  const float2 st = stats[b * G + c / (C / G)];
  float v = (z[i] - st.x) * st.y * gamma[c] + beta[c];
  if (res) v += res[i];
  if (relu) v = fmaxf(v, 0.f);
  z[i] = v;
}

__global__ void maxpool_fp32_kernel(const float* __restrict__ in, float* __restrict__ out, int64_t total, int T_in,
                                    int T_out, int C, int k, int stride, int pad) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total) return;
  const int c = (int)(i % C);
  const int64_t bt = i / C;
  const int t = (int)(bt % T_out);
  const int64_t b = bt / T_out;
  float m = -INFINITY;
  for (int d = 0; d < k; ++d) {
    const int ti = t * stride + d - pad;
    if (ti >= 0 && ti < T_in) m = fmaxf(m, in[(b * T_in + ti) * C + c]);
  }
  out[i] = m;
}

// Global average pool over T, then dot with w[C] + b.  One CTA per window.
template <int IN_DT>
__global__ void __launch_bounds__(256) head_kernel(const void* __restrict__ in, const float* __restrict__ w, float bias,
                                                   int T, int C, float* __restrict__ scores) {
  __shared__ float red[8];
  const int64_t b = blockIdx.x;
  float part = 0.f;
  for (int c = threadIdx.x; c < C; c += blockDim.x) {
    float s = 0.f;
    for (int t = 0; t < T; ++t) s += ld_in<IN_DT>(in, (b * T + t) * (int64_t)C + c);
    part += s * w[c];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
  __syncthreads();
  if (threadIdx.x == 0) {
    float tot = 0.f;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) tot += red[i];
    scores[b] = tot / T + bias;
  }
}

aframe_status af_launch_head(aframe_ctx* ctx, const void* d_in, int in_dt, const float* d_w, float bias, int T, int C,
                             int64_t B, float* d_scores) {
  if (in_dt == AF_DT_F16) head_kernel<AF_DT_F16><<<(unsigned)B, 256, 0, ctx->stream>>>(d_in, d_w, bias, T, C, d_scores);
  else if (in_dt == AF_DT_BF16) head_kernel<AF_DT_BF16><<<(unsigned)B, 256, 0, ctx->stream>>>(d_in, d_w, bias, T, C, d_scores);
  else head_kernel<AF_DT_F32><<<(unsigned)B, 256, 0, ctx->stream>>>(d_in, d_w, bias, T, C, d_scores);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

// ---- slot planning shared by the fp32 and bf16 drivers -------------------------------------------------
bool af_make_plan(const aframe_weights* w, bool fuse_stem_pool, NetPlan& plan) {
  const int n = (int)w->layers.size();
  plan.slot.assign(n, -1);
  plan.elems.assign(n, 0);
  std::vector<int> last_use(n, -1);
  for (int i = 0; i < n; ++i) {
    const LayerDesc& l = w->layers[i];
    if (l.input_from >= 0) last_use[l.input_from] = i;
    if (l.residual_from >= 0) last_use[l.residual_from] = i;
    // a 1x1 projection shortcut may run INSIDE the conv it feeds (conv_tc.cu): that conv then reads the projection's input
    if (l.kind == 0 && l.residual_from >= 0 && w->layers[l.residual_from].kind == 0 && w->layers[l.residual_from].k == 1 &&
        w->layers[l.residual_from].input_from >= 0)
      last_use[w->layers[l.residual_from].input_from] = i;
  }
  std::vector<int> slot_free_at;   // layer index after which the slot is free (-1 = free now)
  plan.n_slots = 0;
  plan.slot_elems = 0;
  for (int i = 0; i < n; ++i) {
    const LayerDesc& l = w->layers[i];
    if (l.kind == 2) continue;   // the head writes scores
    const bool skipped = fuse_stem_pool && l.kind == 0 && i + 1 < n && w->layers[i + 1].kind == 1 &&
                         w->layers[i + 1].input_from == i && last_use[i] == i + 1;
    if (skipped) continue;        // the fused stem kernel never materialises the pre-pool tensor
    plan.elems[i] = (size_t)l.t_out * l.c_out;
    if (plan.elems[i] > plan.slot_elems) plan.slot_elems = plan.elems[i];
    int s = -1;
    for (int j = 0; j < (int)slot_free_at.size(); ++j)
      if (slot_free_at[j] < i) { s = j; break; }
    if (s < 0) { s = (int)slot_free_at.size(); slot_free_at.push_back(0); }
    slot_free_at[s] = last_use[i] < 0 ? i : last_use[i];
    plan.slot[i] = s;
  }
  plan.n_slots = (int)slot_free_at.size();
  return true;
}

aframe_status af_forward_fp32(aframe_ctx* ctx, const aframe_weights* w, const void* d_in, int in_dt, int64_t sB,
                              int64_t sT, const int64_t* choff, int64_t B, float* d_scores) {
  NetPlan plan;
  af_make_plan(w, false, plan);
  const int64_t chunk = 128;
  const size_t slot_bytes = plan.slot_elems * sizeof(float) * (size_t)(B < chunk ? B : chunk);
  const size_t stats_bytes = w->live_gn ? sizeof(float2) * (size_t)chunk * w->n_groups : 0;
  aframe_status st = af_ws_reserve(ctx, ctx->ws_act, slot_bytes * plan.n_slots + stats_bytes);
  if (st != AFRAME_OK) return st;
  char* base = reinterpret_cast<char*>(ctx->ws_act.ptr);
  const int n = (int)w->layers.size();
  for (int64_t b0 = 0; b0 < B; b0 += chunk) {
    const int64_t nb = (B - b0 < chunk) ? (B - b0) : chunk;
    for (int i = 0; i < n; ++i) {
      const LayerDesc& l = w->layers[i];
      const float* src = l.input_from >= 0 ? reinterpret_cast<float*>(base + slot_bytes * plan.slot[l.input_from]) : nullptr;
      float* dst = plan.slot[i] >= 0 ? reinterpret_cast<float*>(base + slot_bytes * plan.slot[i]) : nullptr;
      if (l.kind == 0) {
        ConvArgs a;
        a.w = w->d_w32[i]; a.bias = w->d_bias[i];
        const float* res_ptr = l.residual_from >= 0 ? reinterpret_cast<float*>(base + slot_bytes * plan.slot[l.residual_from]) : nullptr;
        a.res = w->live_gn ? nullptr : res_ptr;          // true GroupNorm: residual and ReLU come after the norm
        a.out = dst; a.rows = nb * l.t_out;
        a.T_in = l.t_in; a.T_out = l.t_out; a.C_in = l.c_in; a.C_out = l.c_out;
        a.k = l.k; a.stride = l.stride; a.pad = l.pad; a.relu = w->live_gn ? 0 : l.relu;
        dim3 grid((unsigned)((a.rows + 63) / 64), (unsigned)((l.c_out + 63) / 64));
        const int pk = l.input_from < 0 ? AFRAME_PROF_STEM : AFRAME_PROF_CONV;
        af_prof_begin(ctx, pk);
        if (l.input_from < 0) {
          const size_t esz = af_dt_bytes(in_dt);
          a.in = reinterpret_cast<const char*>(d_in) + (size_t)(b0 * sB) * esz;
          a.in_sB = sB; a.in_sT = sT; a.in_sC = 0; a.use_choff = 1;
          for (int c = 0; c < AF_MAX_CH; ++c) a.choff[c] = c < l.c_in ? choff[c] : 0;
          if (in_dt == AF_DT_BF16) conv_fp32_kernel<AF_DT_BF16><<<grid, 256, 0, ctx->stream>>>(a);
          else if (in_dt == AF_DT_F16) conv_fp32_kernel<AF_DT_F16><<<grid, 256, 0, ctx->stream>>>(a);
          else conv_fp32_kernel<AF_DT_F32><<<grid, 256, 0, ctx->stream>>>(a);
        } else {
          a.in = src; a.in_sB = (int64_t)l.t_in * l.c_in; a.in_sT = l.c_in; a.in_sC = 1; a.use_choff = 0;
          conv_fp32_kernel<AF_DT_F32><<<grid, 256, 0, ctx->stream>>>(a);
        }
        af_prof_end(ctx, pk, 1);
        AF_LAUNCH_CHECK(ctx);
        if (w->live_gn) {
          float2* stats = reinterpret_cast<float2*>(base + slot_bytes * plan.n_slots);
          gn_stats_kernel<<<dim3((unsigned)nb, (unsigned)w->n_groups), 256, 0, ctx->stream>>>(dst, l.t_out, l.c_out, w->n_groups,
                                                                                             w->gn_eps, stats);
          AF_LAUNCH_CHECK(ctx);
          const int64_t total = nb * l.t_out * l.c_out;
          gn_apply_kernel<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(dst, stats, w->d_gamma[i], w->d_beta[i], res_ptr,
                                                                                    total, l.t_out, l.c_out, w->n_groups, l.relu);
          AF_LAUNCH_CHECK(ctx);
        }
      } else if (l.kind == 1) {
        if (!src) return af_fail(ctx, AFRAME_EUNSUPPORTED, "max-pool directly on the network input is not supported");
        const int64_t total = nb * l.t_out * l.c_out;
        af_prof_begin(ctx, AFRAME_PROF_STEM);
        maxpool_fp32_kernel<<<(unsigned)((total + 255) / 256), 256, 0, ctx->stream>>>(src, dst, total, l.t_in, l.t_out,
                                                                                      l.c_out, l.k, l.stride, l.pad);
        af_prof_end(ctx, AFRAME_PROF_STEM, 1);
        AF_LAUNCH_CHECK(ctx);
      } else {
        if (!src) return af_fail(ctx, AFRAME_EUNSUPPORTED, "head directly on the network input is not supported");
        af_prof_begin(ctx, AFRAME_PROF_HEAD);
        st = af_launch_head(ctx, src, 0, w->d_head_w, w->head_b, l.t_in, l.c_in, nb, d_scores + b0);
        af_prof_end(ctx, AFRAME_PROF_HEAD, 1);
        if (st != AFRAME_OK) return st;
      }
    }
  }
  return AFRAME_OK;
}
