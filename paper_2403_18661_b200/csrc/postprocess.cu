// NEXT-1: "predictions are then integrated over time using a 1 s top hat filter [...] The maximum integrated
// value over an 8 s window is taken as the detection statistic corresponding to a candidate event."
// Readings D1-D3 of DESIGN.md.  Both kernels are pure streaming work (4 B in, 4 B out per score; 12 B per trigger).
#include "common.cuh"

// I[s][i] = mean of scores[s][max(0, i - n_int + 1) .. i], float32 sum in index order, then one multiply (reading D3).
__global__ void __launch_bounds__(256)
tophat_kernel(const float* __restrict__ scores, int64_t n, int64_t ld, int n_int, float* __restrict__ integ, int64_t ld_out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t s = blockIdx.y;
  if (i >= n) return;
  const float* x = scores + s * ld;
  const int64_t lo = i - n_int + 1 > 0 ? i - n_int + 1 : 0;
  float acc = 0.f;
  for (int64_t j = lo; j <= i; ++j) acc = __fadd_rn(acc, x[j]);
  integ[s * ld_out + i] = __fmul_rn(acc, __fdiv_rn(1.0f, (float)(i + 1 - lo)));
}

// One warp per (series, cluster window): first maximum of n_cluster consecutive integrated values.
__global__ void __launch_bounds__(256)
cluster_max_kernel(const float* __restrict__ integ, int64_t n, int64_t ld, int n_cluster, int64_t n_trig,
                   float* __restrict__ trig_value, int64_t* __restrict__ trig_index) {
  const int lane = threadIdx.x & 31;
  const int64_t k = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int64_t s = blockIdx.y;
  if (k >= n_trig) return;
  const int64_t a = k * n_cluster;
  const int64_t b = a + n_cluster < n ? a + n_cluster : n;
  const float* x = integ + s * ld;
  float best = -INFINITY;
  int64_t bi = a;
  bool have = false;
  for (int64_t j = a + lane; j < b; j += 32) {
    const float v = x[j];
    if (!have || v > best) { best = v; bi = j; have = true; }   // NaN never wins; ties keep the earlier index
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, best, o);
    const int64_t oi = __shfl_xor_sync(0xffffffffu, bi, o);
    const int oh = __shfl_xor_sync(0xffffffffu, (int)have, o);
    if (oh && (!have || ov > best || (ov == best && oi < bi))) { best = ov; bi = oi; have = true; }
  }
  if (lane == 0) { trig_value[s * n_trig + k] = best; trig_index[s * n_trig + k] = bi; }
}

AF_API aframe_status aframe_postprocess(aframe_ctx* ctx, const float* d_scores, int64_t n_series, int64_t n, int64_t ld,
                                        int32_t n_int, int32_t n_cluster, float* d_integrated, float* d_trig_value,
                                        int64_t* d_trig_index, int64_t* h_n_trig) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_scores || !d_integrated || !d_trig_value || !d_trig_index || !h_n_trig) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (n_series < 1 || n < 0 || ld < n || n_int < 1 || n_cluster < 1) return af_fail(ctx, AFRAME_EINVAL, "bad size");
  const int64_t n_trig = (n + n_cluster - 1) / n_cluster;
  *h_n_trig = n_trig;
  if (n == 0) return AFRAME_OK;
  tophat_kernel<<<dim3((unsigned)((n + 255) / 256), (unsigned)n_series), 256, 0, ctx->stream>>>(d_scores, n, ld, n_int, d_integrated, n);
  AF_LAUNCH_CHECK(ctx);
  cluster_max_kernel<<<dim3((unsigned)((n_trig + 7) / 8), (unsigned)n_series), 256, 0, ctx->stream>>>(
      d_integrated, n, n, n_cluster, n_trig, d_trig_value, d_trig_index);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
