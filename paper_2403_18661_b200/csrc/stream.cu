// O-6 streaming state (the paper's "snapshotter") and aframe_stream_step.
// Every kernel of an update takes its decisions from a device-resident counter, so the same launch
// sequence (and hence one captured CUDA graph) serves every update.
#include <new>
#include "common.cuh"
#include "stream_net.h"

struct aframe_stream_state {
  aframe_ctx* ctx = nullptr;
  const aframe_weights* w = nullptr;
  int64_t ring_len = 0;
  int n_avg = 0;
  char* blob = nullptr;          // one allocation holding everything below
  size_t blob_bytes = 0;
  int64_t* d_n = nullptr;        // [0] samples received, [1] whitened samples held (<= K)
  int* d_has_filter = nullptr;
  float* d_raw = nullptr;        // [C][ring_len] raw strain ring
  float* d_pgram = nullptr;      // [C][n_avg][F] periodogram ring
  float* d_psd = nullptr;        // [C][F]
  float* d_H = nullptr;          // [C][NOS/2+1] (unused by the FIR update, kept for parity with batch)
  float* d_taps = nullptr;       // [C][L+1]
  float* d_white = nullptr;      // [C][K] newest K whitened samples, oldest first
  float* d_new = nullptr;        // [C][stride]
  af_stream_net* net = nullptr;  // incremental network (stream_net.cu); null: one full forward per update
  // One update = one CUDA graph launch: the launch sequence is captured the first time a given triple of caller
  // pointers is seen and replayed afterwards (every decision of an update is taken on the device from the counters,
  // so the same graph serves every update).  A caller that alternates between a few buffers keeps one graph per triple
  // (least recently used of AF_STREAM_GRAPHS is replaced).
  struct Graph {
    cudaGraphExec_t exec = nullptr;
    const float* in = nullptr; float* scores = nullptr; int32_t* n = nullptr;
    void* ws = nullptr;          // activation workspace the captured launches point into
    int64_t last_use = 0;
  };
  static constexpr int AF_STREAM_GRAPHS = 4;
  Graph graphs[AF_STREAM_GRAPHS];
  int64_t g_launches = 0;        // kernels per replay
  int64_t replays = 0, steps = 0;
};

const aframe_weights* af_stream_weights(const aframe_stream_state* st) { return st->w; }

// Device resources of a state (after the context's stream has been synchronised); the host shell stays valid and dead.
void af_stream_release(aframe_stream_state* st) {
  for (auto& g : st->graphs) { if (g.exec) cudaGraphExecDestroy(g.exec); g = aframe_stream_state::Graph(); }
  cudaFree(st->blob);
  st->blob = nullptr;
  af_stream_net_free(st->net);
  st->net = nullptr;
  cudaGetLastError();
  st->ctx = nullptr; st->w = nullptr;
}

// Append `stride` samples per channel to the ring and advance the counter.  One CTA.
__global__ void stream_ingest_kernel(const float* __restrict__ fresh, int C, int stride, float* __restrict__ raw,
                                     int64_t ring_len, int64_t* __restrict__ d_n) {
  const int64_t n = d_n[0];
  for (int i = threadIdx.x; i < C * stride; i += blockDim.x) {
    const int c = i / stride, t = i - c * stride;
    raw[(int64_t)c * ring_len + (n + t) % ring_len] = fresh[i];
  }
  __syncthreads();
  if (threadIdx.x == 0) d_n[0] = n + stride;
}

// The `stride` newest whitened samples m in [n - s - L/2, n - L/2) by direct summation of the L-1 taps
// (0.52 MMAC per update).  One CTA = FIR_NO consecutive outputs of one channel: the L - 2 + FIR_NO ring samples they
// touch and the taps are staged in shared memory once (ring wrap handled while staging, by a conditional subtract: the
// first version took a 64-bit modulo per tap and cost 36 us of the update), then each warp sums FIR_NO / 8 outputs,
// lane-strided over the taps.
constexpr int FIR_NO = 16;
__global__ void __launch_bounds__(256)
stream_fir_kernel(const float* __restrict__ raw, int64_t ring_len, const float* __restrict__ taps, int L, int stride,
                  float scale, const int64_t* __restrict__ d_n, const int* __restrict__ d_has_filter,
                  float* __restrict__ fresh_white) {
  if (*d_has_filter == 0) return;
  extern __shared__ float fir_smem[];              // [L + 1] taps, then [L - 2 + FIR_NO] samples
  float* hs = fir_smem;
  float* xs = fir_smem + (L + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int o0 = blockIdx.x * FIR_NO;
  const int c = blockIdx.y;
  const int half = L / 2;
  const int64_t n = d_n[0];
  // y[m] = sum_{i = 1}^{L - 1} h[i] x[m + half - i]; outputs m0 + o, o = o0 .. o0 + FIR_NO - 1, read samples
  // m0 + o0 + half - (L - 1) ... m0 + o0 + FIR_NO - 1 + half - 1: xs[k] = x[first + k]
  const int64_t m0 = n - stride - half;
  const int64_t first = m0 + o0 + half - (L - 1);
  const int n_x = L - 2 + FIR_NO;
  const float* x = raw + (int64_t)c * ring_len;
  const float* h = taps + (int64_t)c * (L + 1);
  int64_t p0 = first % ring_len;                    // (one modulo per thread; first >= 0 once a filter exists: n >= psd_len >= stride + L)
  if (p0 < 0) p0 += ring_len;
  for (int k = threadIdx.x; k < n_x; k += 256) {
    int64_t q = p0 + k;
    if (q >= ring_len) q -= ring_len;
    xs[k] = x[q] * scale;
  }
  for (int k = threadIdx.x; k <= L; k += 256) hs[k] = h[k];
  __syncthreads();
  for (int oo = warp; oo < FIR_NO; oo += 8) {
    const int o = o0 + oo;
    if (o >= stride) break;
    // sample of tap i for output oo: x[m0 + o + half - i] = xs[oo + (L - 1) - i]
    float acc0 = 0.f, acc1 = 0.f;
    const float* xo = xs + oo + (L - 1);
    for (int i = 1 + lane; i < L; i += 64) {
      acc0 = fmaf(hs[i], xo[-i], acc0);
      const int i1 = i + 32;
      if (i1 < L) acc1 = fmaf(hs[i1], xo[-i1], acc1);
    }
    float acc = acc0 + acc1;
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, s);
    if (lane == 0) fresh_white[c * stride + o] = acc;
  }
}

// Slide the whitened window by `stride` and append the fresh samples.  One CTA (read all, sync, write).
__global__ void __launch_bounds__(1024)
stream_slide_kernel(float* __restrict__ white, const float* __restrict__ fresh_white, int C, int K, int stride,
                    int64_t* __restrict__ d_n, const int* __restrict__ d_has_filter, int32_t* __restrict__ d_n_scores) {
  if (*d_has_filter == 0) { if (threadIdx.x == 0) *d_n_scores = 0; return; }
  const int total = C * K;
  float v[8];
  int cnt = 0;
  for (int i = threadIdx.x; i < total && cnt < 8; i += blockDim.x, ++cnt) {
    const int c = i / K, t = i - c * K;
    v[cnt] = (t + stride < K) ? white[c * K + t + stride] : fresh_white[c * stride + (t + stride - K)];
  }
  __syncthreads();
  cnt = 0;
  for (int i = threadIdx.x; i < total && cnt < 8; i += blockDim.x, ++cnt) white[i] = v[cnt];
  if (threadIdx.x == 0) {
    int64_t held = d_n[1] + stride;
    if (held > K) held = K;
    d_n[1] = held;
    *d_n_scores = held >= K ? 1 : 0;
  }
}

static size_t align_up(size_t v) { return (v + 255) & ~(size_t)255; }

AF_API aframe_status aframe_stream_reset(aframe_stream_state* st) {
  if (!st || !st->ctx) return AFRAME_ESTATE;
  AF_CUDA(st->ctx, cudaMemsetAsync(st->blob, 0, st->blob_bytes, st->ctx->stream));
  if (st->net) return af_stream_net_reset(st->ctx, st->net);
  return AFRAME_OK;
}

AF_API void aframe_stream_destroy(aframe_stream_state* st) {
  if (!st) return;
  if (aframe_ctx* ctx = st->ctx) {                    // (a dead shell, released with its context or weights, has none)
    cudaStreamSynchronize(ctx->stream);
    for (size_t i = 0; i < ctx->live_streams.size(); ++i)
      if (ctx->live_streams[i] == st) { ctx->live_streams.erase(ctx->live_streams.begin() + i); break; }
    af_stream_release(st);
  }
  delete st;
}

AF_API aframe_status aframe_stream_create(aframe_ctx* ctx, const aframe_weights* w, aframe_stream_state** out) {
  if (!ctx) return AFRAME_EINVAL;
  if (!w || !out) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  *out = nullptr;
  if (w->ctx != ctx) return af_fail(ctx, AFRAME_ESTATE, "weights belong to another context");
  const aframe_config& cfg = ctx->cfg;
  const int C = cfg.n_channels, F = cfg.welch_nfft / 2 + 1, L = cfg.filter_len, K = cfg.kernel_len;
  if ((size_t)C * K > 8 * 1024) return af_fail(ctx, AFRAME_EUNSUPPORTED, "streaming window larger than 8192 samples in total");
  if (cfg.psd_len < cfg.stride + L) return af_fail(ctx, AFRAME_ESHAPE, "psd_len < stride + filter_len");
  // the streaming Welch computes the ONE segment that ends at the newest sample, on the updates where n is a multiple of
  // the hop; with a stride that does not divide the hop some segments would end between updates and never be computed
  if (cfg.welch_hop % cfg.stride) return af_fail(ctx, AFRAME_ESHAPE, "streaming needs welch_hop to be a multiple of stride");
  aframe_stream_state* st = new (std::nothrow) aframe_stream_state();
  if (!st) return af_fail(ctx, AFRAME_ENOMEM, "host allocation failed");
  st->ctx = ctx; st->w = w;
  st->ring_len = cfg.psd_len + cfg.stride;           // trailing psd_len samples + one update of slack
  st->n_avg = (int)((cfg.psd_len - cfg.welch_nfft) / cfg.welch_hop + 1);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  const size_t o_n = take(2 * sizeof(int64_t)), o_f = take(sizeof(int));
  const size_t o_raw = take(sizeof(float) * C * st->ring_len), o_pg = take(sizeof(float) * (size_t)C * st->n_avg * F);
  const size_t o_psd = take(sizeof(float) * C * F), o_H = take(sizeof(float) * C * (AF_NOS / 2 + 1));
  const size_t o_taps = take(sizeof(float) * C * (L + 1)), o_w = take(sizeof(float) * C * K);
  const size_t o_new = take(sizeof(float) * C * cfg.stride);
  st->blob_bytes = off;
  if (cudaMalloc(&st->blob, off) != cudaSuccess) { cudaGetLastError(); delete st; return af_fail(ctx, AFRAME_ENOMEM, "device allocation failed"); }
  st->d_n = reinterpret_cast<int64_t*>(st->blob + o_n);
  st->d_has_filter = reinterpret_cast<int*>(st->blob + o_f);
  st->d_raw = reinterpret_cast<float*>(st->blob + o_raw);
  st->d_pgram = reinterpret_cast<float*>(st->blob + o_pg);
  st->d_psd = reinterpret_cast<float*>(st->blob + o_psd);
  st->d_H = reinterpret_cast<float*>(st->blob + o_H);
  st->d_taps = reinterpret_cast<float*>(st->blob + o_taps);
  st->d_white = reinterpret_cast<float*>(st->blob + o_w);
  st->d_new = reinterpret_cast<float*>(st->blob + o_new);
  // the incremental network where the configuration allows it (cfg.stream_full_forward = 0, folded tensor-core path, a
  // stride that is a multiple of the network's total downsampling and at most 128 samples)
  aframe_status rs = AFRAME_OK;
  if (cfg.stream_full_forward != 1) {
    const char* why = "";
    rs = af_stream_net_create(ctx, w, &st->net, &why);
  }
  if (rs == AFRAME_OK) rs = aframe_stream_reset(st);
  // one untimed forward at B = 1 sizes the activation workspace, builds the tensor maps and sets the
  // kernels' shared-memory attributes, so that aframe_stream_step never allocates (graph capturable)
  float* d_tmp = nullptr;
  if (rs == AFRAME_OK && cudaMalloc(&d_tmp, sizeof(float)) != cudaSuccess) { cudaGetLastError(); rs = AFRAME_ENOMEM; }
  if (rs == AFRAME_OK && !st->net) rs = aframe_forward(ctx, w, st->d_white, 1, d_tmp);
  if (rs == AFRAME_OK && cudaStreamSynchronize(ctx->stream) != cudaSuccess) rs = af_fail(ctx, AFRAME_ECUDA, "stream warm-up forward failed");
  cudaFree(d_tmp);
  if (rs != AFRAME_OK) { cudaGetLastError(); af_stream_release(st); delete st; return rs; }
  ctx->live_streams.push_back(st);
  *out = st;
  return AFRAME_OK;
}

static aframe_status stream_step_enqueue(aframe_ctx* ctx, const float* d_new_samples, aframe_stream_state* st,
                                         float* d_scores, int32_t* d_n_scores);

AF_API int64_t aframe_stream_graph_replays(const aframe_stream_state* st) { return st ? st->replays : 0; }
AF_API int32_t aframe_stream_incremental(const aframe_stream_state* st) { return st && st->net ? af_stream_net_cluster(st->net) : 0; }

AF_API aframe_status aframe_stream_step(aframe_ctx* ctx, const float* d_new_samples, aframe_stream_state* st,
                                        float* d_scores, int32_t* d_n_scores) {
  if (!ctx) return AFRAME_EINVAL;
  if (!st || st->ctx != ctx || !st->w) return af_fail(ctx, AFRAME_ESTATE, "stream state is released (its weights or context are gone) or belongs to another context");
  if (!d_new_samples || !d_scores || !d_n_scores) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(ctx->stream, &cap);
  // direct launches when the caller is capturing the stream itself or when stage timing is on
  // (the legacy default stream cannot be captured: a context bound to it launches directly as well)
  if (ctx->prof_on || ctx->layer_ms || cap != cudaStreamCaptureStatusNone ||
      ctx->stream == nullptr || ctx->stream == cudaStreamLegacy)
    return stream_step_enqueue(ctx, d_new_samples, st, d_scores, d_n_scores);
  // the graph captured for these pointers (a larger forward on the same context may have re-allocated the activation
  // workspace since: then it is stale and captured again)
  st->steps++;
  aframe_stream_state::Graph* hit = nullptr;
  aframe_stream_state::Graph* lru = nullptr;          // an empty slot if there is one, else the least recently used
  for (auto& g : st->graphs) {
    if (g.exec && g.in == d_new_samples && g.scores == d_scores && g.n == d_n_scores) hit = &g;
    if (!lru || (lru->exec && (!g.exec || g.last_use < lru->last_use))) lru = &g;
  }
  if (hit && hit->ws != ctx->ws_act.ptr) { lru = hit; hit = nullptr; }
  if (!hit) {
    if (lru->exec) {                                  // (it may still be in flight)
      AF_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
      cudaGraphExecDestroy(lru->exec);
      *lru = aframe_stream_state::Graph();
    }
    const int64_t l0 = ctx->launches;
    AF_CUDA(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
    aframe_status rs = stream_step_enqueue(ctx, d_new_samples, st, d_scores, d_n_scores);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(ctx->stream, &g);
    st->g_launches = ctx->launches - l0;
    ctx->launches = l0;
    if (rs != AFRAME_OK) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return rs; }
    if (e != cudaSuccess || !g) { cudaGetLastError(); return af_fail(ctx, AFRAME_ECUDA, "stream capture failed: %s", cudaGetErrorString(e)); }
    e = cudaGraphInstantiate(&lru->exec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { lru->exec = nullptr; cudaGetLastError(); return af_fail(ctx, AFRAME_ECUDA, "graph instantiation failed: %s", cudaGetErrorString(e)); }
    lru->in = d_new_samples; lru->scores = d_scores; lru->n = d_n_scores;
    lru->ws = ctx->ws_act.ptr;
    hit = lru;
  }
  hit->last_use = st->steps;
  AF_CUDA(ctx, cudaGraphLaunch(hit->exec, ctx->stream));
  ctx->launches += st->g_launches;
  st->replays++;
  return AFRAME_OK;
}

static aframe_status stream_step_enqueue(aframe_ctx* ctx, const float* d_new_samples, aframe_stream_state* st,
                                         float* d_scores, int32_t* d_n_scores) {
  const aframe_config& cfg = ctx->cfg;
  const int C = cfg.n_channels, L = cfg.filter_len, K = cfg.kernel_len, s = cfg.stride;
  stream_ingest_kernel<<<1, 256, 0, ctx->stream>>>(d_new_samples, C, s, st->d_raw, st->ring_len, st->d_n);
  AF_LAUNCH_CHECK(ctx);
  StreamGate gate;
  gate.d_n = st->d_n; gate.d_has_filter = st->d_has_filter; gate.ring_len = st->ring_len;
  gate.psd_len = cfg.psd_len; gate.psd_update = cfg.psd_update;
  aframe_status rs = af_launch_welch_periodograms(ctx, st->d_raw, st->ring_len, 0, st->n_avg, st->d_pgram, &gate);
  if (rs != AFRAME_OK) return rs;
  rs = af_launch_psd_mean(ctx, st->d_pgram, st->n_avg, 0, 1, st->n_avg, st->d_psd, &gate);
  if (rs != AFRAME_OK) return rs;
  rs = af_launch_filter_design(ctx, st->d_psd, 1, st->d_H, st->d_taps, &gate);
  if (rs != AFRAME_OK) return rs;
  const float scale = ldexpf(1.0f, cfg.strain_scale_log2);
  stream_fir_kernel<<<dim3((unsigned)((s + FIR_NO - 1) / FIR_NO), (unsigned)C), 256, sizeof(float) * (2 * L - 1 + FIR_NO), ctx->stream>>>(
      st->d_raw, st->ring_len, st->d_taps, L, s, scale, st->d_n, st->d_has_filter, st->d_new);
  AF_LAUNCH_CHECK(ctx);
  stream_slide_kernel<<<1, 1024, 0, ctx->stream>>>(st->d_white, st->d_new, C, K, s, st->d_n, st->d_has_filter, d_n_scores);
  AF_LAUNCH_CHECK(ctx);
  if (st->net) return af_stream_net_launch(ctx, st->net, st->d_white, st->d_n, st->d_has_filter, d_n_scores, d_scores);
  return aframe_forward(ctx, st->w, st->d_white, 1, d_scores);
}
