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

// (value, index) order of the clustering: a NaN beats every number (NaN propagates: the trigger of a window that holds
// one is its FIRST NaN, as numpy.argmax gives for the oracle); among equals the earlier index wins.
__device__ __forceinline__ bool cluster_better(float v, int64_t vi, float b, int64_t bi) {
  const bool vn = v != v, bn = b != b;
  if (vn != bn) return vn;
  if (vn) return vi < bi;
  return v > b || (v == b && vi < bi);
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
    if (!have || cluster_better(v, j, best, bi)) { best = v; bi = j; have = true; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, best, o);
    const int64_t oi = __shfl_xor_sync(0xffffffffu, bi, o);
    const int oh = __shfl_xor_sync(0xffffffffu, (int)have, o);
    if (oh && (!have || cluster_better(ov, oi, best, bi))) { best = ov; bi = oi; have = true; }
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

// NEXT-4: "a false alarm rate (FAR) can be assigned to injected events by dividing the number of
// background events with detection statistic greater than the event of interest, with livetime analyzed."
// counts[i] = #{b : background[b] > events[i]}: an exact integer, so no sort is needed -- a tiled all-pairs compare.
// Grid (event tiles, background chunks).  A thread keeps FAR_EV events in registers; the CTA streams its background
// chunk through shared memory (every lane reads the same float4: a broadcast) and adds its partial counts with one
// atomic per event.  2 instructions per pair; 1e7 background x 1e4 events is a few milliseconds.
constexpr int FAR_EV = 4;            // events per thread
constexpr int FAR_THREADS = 256;
constexpr int FAR_STAGE = 2048;      // background values per shared-memory stage
constexpr int FAR_CHUNK = 16 * FAR_STAGE;

__global__ void __launch_bounds__(FAR_THREADS)
far_count_kernel(const float* __restrict__ bg, int64_t n_bg, const float* __restrict__ ev, int64_t n_ev,
                 unsigned long long* __restrict__ counts) {
  __shared__ __align__(16) float sb[FAR_STAGE];
  const int tid = threadIdx.x;
  const int64_t e0 = ((int64_t)blockIdx.x * FAR_THREADS + tid) * FAR_EV;
  float e[FAR_EV];
  unsigned int n[FAR_EV];
#pragma unroll
  for (int k = 0; k < FAR_EV; ++k) { e[k] = e0 + k < n_ev ? ev[e0 + k] : INFINITY; n[k] = 0u; }
  const int64_t c0 = (int64_t)blockIdx.y * FAR_CHUNK;
  const int64_t c1 = c0 + FAR_CHUNK < n_bg ? c0 + FAR_CHUNK : n_bg;
  for (int64_t s0 = c0; s0 < c1; s0 += FAR_STAGE) {
    __syncthreads();
    for (int i = tid; i < FAR_STAGE; i += FAR_THREADS) sb[i] = s0 + i < c1 ? bg[s0 + i] : -INFINITY;   // padding never counts
    __syncthreads();
#pragma unroll 4
    for (int i = 0; i < FAR_STAGE; i += 4) {
      const float4 b = *reinterpret_cast<const float4*>(&sb[i]);
#pragma unroll
      for (int k = 0; k < FAR_EV; ++k)
        n[k] += (unsigned)(b.x > e[k]) + (unsigned)(b.y > e[k]) + (unsigned)(b.z > e[k]) + (unsigned)(b.w > e[k]);
    }
  }
#pragma unroll
  for (int k = 0; k < FAR_EV; ++k)
    if (e0 + k < n_ev && n[k]) atomicAdd(&counts[e0 + k], (unsigned long long)n[k]);
}

__global__ void far_rate_kernel(const long long* __restrict__ counts, int64_t n_ev, double livetime_s, double* __restrict__ far) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_ev) far[i] = __ddiv_rn((double)counts[i], livetime_s);
}

AF_API aframe_status aframe_far(aframe_ctx* ctx, const float* d_background, int64_t n_bg, const float* d_events,
                                int64_t n_ev, double livetime_s, int64_t* d_counts, double* d_far) {
  if (!ctx) return AFRAME_EINVAL;
  if (n_bg < 0 || n_ev < 0) return af_fail(ctx, AFRAME_EINVAL, "negative size");
  if (n_ev == 0) return AFRAME_OK;
  if (!d_events || !d_counts || (n_bg > 0 && !d_background)) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (d_far && !(livetime_s > 0.0)) return af_fail(ctx, AFRAME_EINVAL, "livetime_s must be positive");
  AF_CUDA(ctx, cudaMemsetAsync(d_counts, 0, sizeof(int64_t) * (size_t)n_ev, ctx->stream));
  if (n_bg > 0) {
    const int64_t ev_tiles = (n_ev + FAR_THREADS * FAR_EV - 1) / (FAR_THREADS * FAR_EV);
    const int64_t bg_chunks = (n_bg + FAR_CHUNK - 1) / FAR_CHUNK;
    if (bg_chunks > 65535) return af_fail(ctx, AFRAME_ESHAPE, "far: more than 65535 * 32768 background values");
    far_count_kernel<<<dim3((unsigned)ev_tiles, (unsigned)bg_chunks), FAR_THREADS, 0, ctx->stream>>>(
        d_background, n_bg, d_events, n_ev, reinterpret_cast<unsigned long long*>(d_counts));
    AF_LAUNCH_CHECK(ctx);
  }
  if (d_far) {
    far_rate_kernel<<<(unsigned)((n_ev + 255) / 256), 256, 0, ctx->stream>>>(reinterpret_cast<const long long*>(d_counts), n_ev,
                                                                           livetime_s, d_far);
    AF_LAUNCH_CHECK(ctx);
  }
  return AFRAME_OK;
}
