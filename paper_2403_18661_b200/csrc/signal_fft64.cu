// Overlap-save whitening, paired Welch periodograms and the plain batched rFFT / irFFT on the 64 x 64 register transform
// of fft64.cuh.
//
//  O-3 ("whitened in the frequency-domain, and transformed back to time-domain")   whiten_os64_kernel
//  O-1 (reading A1)                                                               welch_pair_kernel
//  the standalone transform BASELINE.json's north_star names (measurement hook)                 rfft64_kernel, irfft64_kernel
//
// One transform = 64 threads (two warps) with 64 complex elements each.  A CTA of 128 threads runs two independent
// transforms (sub-block g = tid / 64; with two detectors: the two channels of one overlap-save block), synchronised by
// the named barriers 1 + g, and walks its work items persistently so the 32 KB twiddle table is built once per CTA.
#include "fft64.cuh"
#include <atomic>

constexpr int W64_M = 4096;                       // complex length = AF_NOS / 2
constexpr int W64_THREADS = 128;
constexpr size_t W64_SMEM = sizeof(float2) * (2 * F64_TILE + 4096);
static_assert(AF_NOS == 2 * W64_M, "the 64 x 64 transform is built for 8192-sample overlap-save blocks");

// ---- the real-input transform pair around a spectral operation -------------------------------------------------------
// Forward: the block's 8192 real samples are read as 4096 complex z[n] = x[2n] + i x[2n+1]; after two passes thread t
// holds Z[t + 64 k2] in v[k2].  The spectrum of the real block, X[k] = E[k] + W_8192^k O[k] with E = (Z[k] + conj Z[M-k])/2,
// O = -i (Z[k] - conj Z[M-k])/2, needs the mirror element, which lives in thread (64 - t) & 63 at k2' = 63 - k2 (thread 0:
// (64 - k2) & 63).  Every thread therefore handles the 32 pairs (k, M - k) of its LOWER half k2 < 32: it fetches the mirror
// elements from its partner's upper half through shared memory, computes both results of the pair, keeps its own and hands
// the mirror's result back the same way.  (k = 0 pairs with itself and yields DC and Nyquist; k = M/2, thread 0's k2 = 32,
// is its own mirror and is patched by thread 0.)

// Mirror exchange, part 1: publish the upper half (and element 0, thread 0's own mirror).
__device__ __forceinline__ void mirror_publish(const float2 (&v)[64], float2* tile, int t, int bar) {
  tile[t * F64_ROW] = v[0];
#pragma unroll
  for (int k2 = 32; k2 < 64; ++k2) tile[t * F64_ROW + k2] = v[k2];
  f64_bar(bar);
}
// shared-memory slot of the mirror of (t, k2), k2 < 32: read from there, and its result goes back there
__device__ __forceinline__ float2* mirror_slot(float2* tile, int t, int k2) {
  const int p = (64 - t) & 63, z = t == 0 ? 1 : 0;
  return tile + p * F64_ROW + (k2 == 0 ? (z ? 0 : 63) : 63 + z - k2);
}

// --------------------------------------------------------------------------------------------------
// Overlap-save whitening.  Work item = (overlap-save block, channel).
// --------------------------------------------------------------------------------------------------
template <int OUT_DT>
__global__ void __launch_bounds__(W64_THREADS, 2)
whiten_os64_kernel(const float* __restrict__ strain, int64_t n_samples, int64_t ld, const float* __restrict__ H, int C,
                   int64_t in0, int64_t out_total, int64_t epoch_len, int blocks_per_epoch, int64_t n_items, int L, float scale,
                   const float2* __restrict__ tw, void* __restrict__ out_v, int64_t ld_out) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tab = reinterpret_cast<float2*>(smem_raw);
  const int tid = threadIdx.x, g = tid >> 6, t = tid & 63;
  float2* tile = tab + 4096 + g * F64_TILE;
  f64_fill_tab(tab, tw, tid, W64_THREADS);
  __syncthreads();
  const int bar = 1 + g;
  const int valid = AF_NOS - L, half = L / 2;
  const float2 wt = __ldg(tw + t);               // W_8192^t
  constexpr int M = W64_M;

  for (int64_t item = (int64_t)blockIdx.x * 2 + g; item < n_items; item += (int64_t)gridDim.x * 2) {
    const int c = (int)(item % C);
    const int64_t bi = item / C;
    const int64_t e = bi / blocks_per_epoch;
    const int sb = (int)(bi - e * blocks_per_epoch);
    const int64_t out0 = e * epoch_len + (int64_t)sb * valid;
    int64_t n_valid = epoch_len - (int64_t)sb * valid;
    if (n_valid > valid) n_valid = valid;
    if (n_valid > out_total - out0) n_valid = out_total - out0;
    if (n_valid <= 0) continue;                  // (uniform over the 64 threads of the transform)
    const int64_t x0 = in0 + out0;
    const float* x = strain + (int64_t)c * ld + x0;
    const float* Hc = H + (e * C + c) * (int64_t)(M + 1);

    // Four 64-point register transforms per item, ONE copy of their code: the pass loop is kept rolled (the unrolled kernel
    // was 180 KB of straight-line code and spent 2.4 cycles waiting for instructions per instruction issued).  The inverse
    // transform runs through the same forward code on conjugated data (IFFT(y) = conj(FFT(conj(y)))).
    // the item's transfer-function values are read once, by one thread each: fetched into L1 now, they are there when the
    // spectral multiply needs them (2 x 32 lines of H[k], 2 x 32 of H[M - k]); the next item's samples go to L2 meanwhile
    {
      const float* hp = Hc + (t < 32 ? 0 : M + 1 - 2048) + (t & 31) * 64 + (t < 32 ? 0 : -1);
      asm volatile("prefetch.global.L1 [%0];" ::"l"(hp < Hc ? Hc : hp));
      asm volatile("prefetch.global.L1 [%0];" ::"l"(hp + 32));
      const int64_t nxt = item + (int64_t)gridDim.x * 2;
      if (nxt < n_items) {
        const int64_t bn = nxt / C, en = bn / blocks_per_epoch;
        const float* xn = strain + (nxt % C) * ld + in0 + en * epoch_len + (bn - en * blocks_per_epoch) * (int64_t)valid;
#pragma unroll
        for (int j = 0; j < 4; ++j) asm volatile("prefetch.global.L2 [%0];" ::"l"(xn + (j * 64 + t) * 32));
      }
    }
    float2 v[64];
    const bool vec_ok = ((reinterpret_cast<uintptr_t>(x) & 7) == 0) && (x0 + AF_NOS <= n_samples);
    const int64_t lim = n_samples - x0;          // samples of this block that exist (the rest reads as zero)
    const int nv = (int)n_valid;
#pragma unroll 1
    for (int pass = 0; pass < 4; ++pass) {
      if (pass == 0) {
        // the block's 8192 real samples as 4096 complex z[n] = x[2n] + i x[2n+1]; thread t takes n = t + 64 n1
        if (vec_ok) {
          const float2* x2 = reinterpret_cast<const float2*>(x);
#pragma unroll
          for (int b = 0; b < 8; ++b)            // (in the order the first butterflies consume them)
#pragma unroll
            for (int a = 0; a < 8; ++a) v[8 * a + b] = __ldg(x2 + 64 * (8 * a + b) + t);
        } else {                                 // ragged or unaligned block (rare): staged through the tile by a rolled loop
          for (int n = t; n < M; n += 64)
            tile[(n >> 6) * F64_ROW + (n & 63)] = make_float2(2 * n < lim ? x[2 * n] : 0.f, 2 * n + 1 < lim ? x[2 * n + 1] : 0.f);
#pragma unroll
          for (int n1 = 0; n1 < 64; ++n1) v[n1] = tile[n1 * F64_ROW + t];   // (its own writes: no barrier needed)
          f64_bar(bar);                          // ... but every thread has read before the first pass stores into the tile
        }
      } else if (pass & 1) {
        f64_load_row(v, tile, t);
      }
      fft64<-1>(v);
      if (!(pass & 1)) {
        f64_twiddle_store<-1>(v, tile, tab, t);
        f64_bar(bar);
      } else if (pass == 1) {
        // spectral multiply by the real transfer function (O-3): Y[k] = H[k] X[k], Y[M - k] = H[M - k] X[M - k], then back to
        // the packed form Z'[k] = (Y_E + i Y_O)[k], kept CONJUGATED for the inverse.  The 2^70 strain scale (reading A9) and
        // the four halves of E, O, Y_E, Y_O ride on H.
        mirror_publish(v, tile, t, bar);
        const float hs = 0.25f * scale;
#pragma unroll
        for (int k0 = 0; k0 < 32; k0 += 8) {     // eight pairs at a time (register pressure)
          float2 zm[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) zm[j] = *mirror_slot(tile, t, k0 + j);
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int k2 = k0 + j;
            const int k = t + 64 * k2;
            const float2 w = f64_cmul_cs<-1>(wt, w128_cs(k2));   // W_8192^k = W_8192^t W_128^k2
            const float hk = __ldg(Hc + k) * hs, hm = __ldg(Hc + M - k) * hs;
            const float2 zk = v[k2], zq = zm[j];
            const float2 ee = make_float2(zk.x + zq.x, zk.y - zq.y);          // 2 E
            const float2 oo = make_float2(zk.y + zq.y, zq.x - zk.x);          // 2 O
            const float2 wo = f64_cmul<false>(oo, w);
            const float2 yk = make_float2(hk * (ee.x + wo.x), hk * (ee.y + wo.y));   // Y[k] / 2
            const float2 ym = make_float2(hm * (ee.x - wo.x), hm * (ee.y - wo.y));   // conj(Y[M - k]) / 2
            const float2 ep = make_float2(yk.x + ym.x, yk.y + ym.y);
            const float2 op = f64_cmul<true>(make_float2(yk.x - ym.x, yk.y - ym.y), w);
            v[k2] = make_float2(ep.x - op.y, -(ep.y + op.x));                        // conj(Z'[k]),  Z'[k] = E' + i O'
            *mirror_slot(tile, t, k2) = make_float2(ep.x + op.y, ep.y - op.x);       // conj(Z'[M - k]), Z'[M - k] = conj(E') + i conj(O')
          }
        }
        f64_bar(bar);
#pragma unroll
        for (int k2 = 32; k2 < 64; ++k2) v[k2] = tile[t * F64_ROW + k2];
        if (t == 0) {                            // k = M/2 is its own mirror: Z'[M/2] = H[M/2] Z[M/2]
          const float h = __ldg(Hc + M / 2) * scale;
          v[32] = make_float2(v[32].x * h, -(v[32].y * h));
        }
        f64_bar(bar);                            // every row has been read back before the next pass overwrites the tile
      } else {
        // v[n1] = conj(z[t + 64 n1]): x[2n] = Re z[n], x[2n+1] = Im z[n] (1/M rides on H); valid outputs are i = 2n - L/2 in
        // [0, n_valid): one vector store per element where both samples are valid and the address is aligned, else the (at
        // most two) ragged positions alone
        constexpr int ESZ = OUT_DT == AF_DT_F32 ? 4 : 2;
        unsigned char* o = reinterpret_cast<unsigned char*>(out_v) + ((int64_t)c * ld_out + out0) * ESZ;
        auto cvt1 = [](float a) -> uint16_t {
          if (OUT_DT == AF_DT_BF16) return __bfloat16_as_ushort(__float2bfloat16_rn(a));
          return (uint16_t)(af_act_pack2(a, 0.f) & 0xffffu);
        };
        const bool st_vec = ((reinterpret_cast<uintptr_t>(o) & (2 * ESZ - 1)) == 0) && ((half & 1) == 0) && ((nv & 1) == 0);
        if (st_vec) {
#pragma unroll
          for (int n1 = 0; n1 < 64; ++n1) {
            const int i0 = 2 * (t + 64 * n1) - half;
            const float a = v[n1].x, b = -v[n1].y;
            if ((unsigned)i0 < (unsigned)nv) {
              if (OUT_DT == AF_DT_F32) *reinterpret_cast<float2*>(o + (int64_t)i0 * ESZ) = make_float2(a, b);
              else if (OUT_DT == AF_DT_BF16) *reinterpret_cast<uint32_t*>(o + (int64_t)i0 * ESZ) = (uint32_t)cvt1(a) | ((uint32_t)cvt1(b) << 16);
              else *reinterpret_cast<uint32_t*>(o + (int64_t)i0 * ESZ) = af_act_pack2(a, b);
            }
          }
        } else {                                 // unaligned output or an odd count (rare): through the tile, scalar stores
          f64_bar(bar);
#pragma unroll
          for (int n1 = 0; n1 < 64; ++n1) tile[n1 * F64_ROW + t] = make_float2(v[n1].x, -v[n1].y);
          f64_bar(bar);
          for (int i = t; i < nv; i += 64) {
            const int s2 = i + half, n = s2 >> 1;
            const float2 zz = tile[(n >> 6) * F64_ROW + (n & 63)];
            const float val = (s2 & 1) ? zz.y : zz.x;
            if (OUT_DT == AF_DT_F32) reinterpret_cast<float*>(o)[i] = val;
            else reinterpret_cast<uint16_t*>(o)[i] = cvt1(val);
          }
        }
      }
    }
    f64_bar(bar);                                // the tile is free for the next item's first pass
  }
}

template <typename K> static aframe_status w64_set_smem(aframe_ctx* ctx, K kern, std::atomic<uint64_t>& done) {
  const uint64_t bit = 1ull << (ctx->device & 63);
  if (!(done.load(std::memory_order_acquire) & bit)) {
    AF_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)W64_SMEM));
    done.fetch_or(bit, std::memory_order_release);
  }
  return AFRAME_OK;
}

aframe_status af_launch_whiten_os(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                  const float* d_H, int64_t in0, int64_t out_total, int64_t epoch_len, int64_t n_epochs,
                                  void* d_out, int64_t ld_out, int out_dt) {
  if (out_total <= 0 || n_epochs <= 0) return AFRAME_OK;
  const aframe_config& cfg = ctx->cfg;
  const int valid = AF_NOS - cfg.filter_len;
  const int bpe = (int)((epoch_len + valid - 1) / valid);
  const float scale = ldexpf(1.0f, cfg.strain_scale_log2);
  const int C = af_nch(ctx);
  const int64_t n_items = n_epochs * bpe * C;
  const int64_t want = (n_items + 1) / 2, cap = 2 * (int64_t)ctx->n_sms;     // two resident CTAs per SM, persistent
  dim3 grid((unsigned)(want < cap ? want : cap));
  af_prof_begin(ctx, AFRAME_PROF_WHITEN);
#define AF_W64_LAUNCH(DT)                                                                                              \
  do {                                                                                                                 \
    static std::atomic<uint64_t> done{0};                                                                              \
    aframe_status st_ = w64_set_smem(ctx, whiten_os64_kernel<DT>, done);                                               \
    if (st_ != AFRAME_OK) return st_;                                                                                  \
    whiten_os64_kernel<DT><<<grid, W64_THREADS, W64_SMEM, ctx->stream>>>(d_strain, n_samples, ld, d_H, C, in0, out_total, \
                                                                        epoch_len, bpe, n_items, cfg.filter_len, scale,   \
                                                                        ctx->d_tw32, d_out, ld_out);                      \
  } while (0)
  if (out_dt == AF_DT_BF16) AF_W64_LAUNCH(AF_DT_BF16);
  else if (out_dt == AF_DT_F16) AF_W64_LAUNCH(AF_DT_F16);
  else AF_W64_LAUNCH(AF_DT_F32);
#undef AF_W64_LAUNCH
  af_prof_end(ctx, AFRAME_PROF_WHITEN, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

// --------------------------------------------------------------------------------------------------
// Welch periodograms of a stored record, two segments per transform (welch_nfft = 4096 only).
// Segments 2q and 2q + 1 (50 % overlap: they share 2048 samples) are mean-detrended, Hann-windowed and transformed
// TOGETHER as z = a + i b; their spectra are A[k] = (Z[k] + conj Z[N-k]) / 2, B[k] = (Z[k] - conj Z[N-k]) / (2 i), and only the
// squared magnitudes are needed: no untangling multiply.  Work item = (segment pair, channel).
// --------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(W64_THREADS, 2)
welch_pair_kernel(const float* __restrict__ strain, int64_t ld, int64_t n_seg, int64_t seg_stride_out, int C, int64_t n_items,
                  float scale, float norm, const float2* __restrict__ tw, float* __restrict__ pgram) {
  constexpr int N = 4096, HOP = 2048, F = N / 2 + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tab = reinterpret_cast<float2*>(smem_raw);
  const int tid = threadIdx.x, g = tid >> 6, t = tid & 63, lane = tid & 31, wq = (tid >> 5) & 1;
  float2* tile = tab + 4096 + g * F64_TILE;
  __shared__ float2 red[2][2];
  f64_fill_tab(tab, tw, tid, W64_THREADS);
  __syncthreads();
  const int bar = 1 + g;
  const float2 wt = __ldg(tw + 2 * t);           // (cos, -sin)(2 pi t / 4096)
  const int64_t n_pairs = (n_seg + 1) / 2;

  for (int64_t item = (int64_t)blockIdx.x * 2 + g; item < n_items; item += (int64_t)gridDim.x * 2) {
    const int c = (int)(item % C);
    const int64_t q = item / C;
    const bool has_b = 2 * q + 1 < n_seg;
    const float* x = strain + (int64_t)c * ld + 2 * q * HOP;
    // thread t holds samples 64 m + t of the 6144 the pair covers: a[n1] = X[n1], b[n1] = X[n1 + 32]
    float xs[96];
#pragma unroll
    for (int m = 0; m < 64; ++m) xs[m] = __ldg(x + 64 * m + t) * scale;
#pragma unroll
    for (int m = 64; m < 96; ++m) xs[m] = has_b ? __ldg(x + 64 * m + t) * scale : 0.f;
    // detrend = 'constant' (reading A1): each segment's own mean
    float sa = 0.f, sm = 0.f, sb = 0.f;
#pragma unroll
    for (int m = 0; m < 32; ++m) { sa += xs[m]; sm += xs[m + 32]; sb += xs[m + 64]; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      sa += __shfl_xor_sync(0xffffffffu, sa, o); sm += __shfl_xor_sync(0xffffffffu, sm, o); sb += __shfl_xor_sync(0xffffffffu, sb, o);
    }
    if (lane == 0) red[g][wq] = make_float2(sa + sm, sm + sb);
    f64_bar(bar);
    const float mean_a = (red[g][0].x + red[g][1].x) * (1.0f / N), mean_b = (red[g][0].y + red[g][1].y) * (1.0f / N);
    // periodic Hann w[n] = 0.5 - 0.5 cos(2 pi n / 4096), n = 64 n1 + t: cos(u + v) with u = 2 pi n1 / 64 a constant
    float2 v[64];
#pragma unroll
    for (int n1 = 0; n1 < 64; ++n1) {
      const float2 cs = w64_cs(n1);
      const float w = fmaf(-0.5f * cs.x, wt.x, fmaf(-0.5f * cs.y, wt.y, 0.5f));   // wt.y = -sin
      v[n1] = make_float2((xs[n1] - mean_a) * w, has_b ? (xs[n1 + 32] - mean_b) * w : 0.f);
    }
    fft64<-1>(v);
    f64_twiddle_store<-1>(v, tile, tab, t);
    f64_bar(bar);
    f64_load_row(v, tile, t);
    fft64<-1>(v);
    mirror_publish(v, tile, t, bar);
    float* oa = pgram + ((int64_t)c * seg_stride_out + 2 * q) * F;
    float* ob = oa + F;
#pragma unroll
    for (int k2 = 0; k2 < 32; ++k2) {
      const float2 zk = v[k2], zq = *mirror_slot(tile, t, k2);
      const float ar = zk.x + zq.x, ai = zk.y - zq.y, br = zk.x - zq.x, bi = zk.y + zq.y;
      const float nk = (k2 == 0 && t == 0) ? 0.25f * norm : 0.5f * norm;           // one-sided: doubled except k = 0, N/2
      const int k = t + 64 * k2;
      oa[k] = (ar * ar + ai * ai) * nk;
      if (has_b) ob[k] = (br * br + bi * bi) * nk;
    }
    if (t == 0) {                                // k = N/2 is its own mirror: A = Re Z, B = Im Z
      oa[N / 2] = v[32].x * v[32].x * norm;
      if (has_b) ob[N / 2] = v[32].y * v[32].y * norm;
    }
    f64_bar(bar);                                // the tile and `red` are free for the next item
  }
  (void)n_pairs;
}

// G[c][j][k] = sum of the `step` consecutive periodograms j step .. j step + step - 1, and Tl[c][j][k] = the sum of the first
// step - 1 of them (the same additions in the same order, one term earlier).  fp32: a sum of n_avg = 63 positive terms taken
// as 7 group sums of 8 plus 7 single terms is good to a few 1e-7 relative, against the 1e-4 of rule T1.
__global__ void psd_group_sum_kernel(const float* __restrict__ pgram, int64_t n_seg_total, int step, int64_t n_groups, int F,
                                     float* __restrict__ G, float* __restrict__ Tl) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t j = blockIdx.y;
  const int c = blockIdx.z;
  if (k >= F) return;
  const float* p = pgram + ((int64_t)c * n_seg_total + j * step) * F + k;
  float acc = 0.f, head = 0.f;
#pragma unroll 8
  for (int i = 0; i < step; ++i, p += F) {
    if (i == step - 1) head = acc;
    acc += *p;
  }
  G[((int64_t)c * n_groups + j) * F + k] = acc;
  Tl[((int64_t)c * n_groups + j) * F + k] = head;
}
// PSD of epoch e = mean of the n_avg periodograms from segment e step on = (n_avg / step whole groups + the rest) / n_avg.
// rest == step - 1 (63 = 7 x 8 + 7): the rest is Tl of the next group -- 8 reads per bin instead of 14, none of them from
// the periodograms; else the single terms are read.
__global__ void psd_mean_grouped_kernel(const float* __restrict__ pgram, const float* __restrict__ G, const float* __restrict__ Tl,
                                        int64_t n_seg_total, int64_t n_groups, int step, int n_avg, int F, int C, float inv_n,
                                        float* __restrict__ psd) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t e = blockIdx.y;
  const int c = blockIdx.z;
  if (k >= F) return;
  const int n_full = n_avg / step, n_rest = n_avg - n_full * step;
  const float* gp = G + ((int64_t)c * n_groups + e) * F + k;
  float a0 = 0.f, a1 = 0.f;
#pragma unroll 8
  for (int j = 0; j < n_full; ++j, gp += F) a0 += *gp;
  if (n_rest == step - 1 && e + n_full < n_groups) {
    a1 = Tl[((int64_t)c * n_groups + e + n_full) * F + k];
  } else {
    const float* p = pgram + ((int64_t)c * n_seg_total + e * step + (int64_t)n_full * step) * F + k;
#pragma unroll 8
    for (int i = 0; i < n_rest; ++i, p += F) a1 += *p;
  }
  psd[((int64_t)e * C + c) * F + k] = (a0 + a1) * inv_n;
}

static std::atomic<uint64_t> g_welch_pair_attr{0};

// Periodograms of segments [0, n_seg) of a stored record (welch_nfft 4096): returns false if this path does not apply.
bool af_welch_pair_applicable(const aframe_ctx* ctx, int64_t n_seg) {
  return ctx->cfg.welch_nfft == 4096 && ctx->cfg.welch_hop == 2048 && n_seg >= 2;
}
aframe_status af_launch_welch_pairs(aframe_ctx* ctx, const float* d_strain, int64_t ld, int64_t n_seg, float* d_pgram) {
  const aframe_config& cfg = ctx->cfg;
  const int C = af_nch(ctx);
  const float scale = ldexpf(1.0f, cfg.strain_scale_log2);
  const float norm = (float)(1.0 / (cfg.fs * 0.375 * cfg.welch_nfft));   // 1 / (fs sum w^2), periodic Hann
  const int64_t n_items = ((n_seg + 1) / 2) * C;
  const int64_t want = (n_items + 1) / 2, cap = 2 * (int64_t)ctx->n_sms;
  aframe_status st = w64_set_smem(ctx, welch_pair_kernel, g_welch_pair_attr);
  if (st != AFRAME_OK) return st;
  af_prof_begin(ctx, AFRAME_PROF_WELCH);
  welch_pair_kernel<<<(unsigned)(want < cap ? want : cap), W64_THREADS, W64_SMEM, ctx->stream>>>(
      d_strain, ld, n_seg, n_seg, C, n_items, scale, norm, ctx->d_tw32, d_pgram);
  af_prof_end(ctx, AFRAME_PROF_WELCH, 1);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

// Mean PSD per epoch through group sums (reads n_avg / step + n_avg % step values per bin and epoch instead of n_avg).
// d_groups: scratch of 2 * C * n_groups * F floats, n_groups = n_seg_total / step.
aframe_status af_launch_psd_mean_grouped(aframe_ctx* ctx, const float* d_pgram, int64_t n_seg_total, int64_t seg_step,
                                         int64_t n_epochs, int64_t n_avg, float* d_groups, float* d_psd) {
  const int F = ctx->cfg.welch_nfft / 2 + 1, C = af_nch(ctx);
  const int64_t n_groups = n_seg_total / seg_step;
  af_prof_begin(ctx, AFRAME_PROF_WELCH);
  float* d_tails = d_groups + (size_t)C * n_groups * F;            // (the caller reserves both halves)
  psd_group_sum_kernel<<<dim3((F + 127) / 128, (unsigned)n_groups, (unsigned)C), 128, 0, ctx->stream>>>(
      d_pgram, n_seg_total, (int)seg_step, n_groups, F, d_groups, d_tails);
  AF_LAUNCH_CHECK(ctx);
  psd_mean_grouped_kernel<<<dim3((F + 127) / 128, (unsigned)n_epochs, (unsigned)C), 128, 0, ctx->stream>>>(
      d_pgram, d_groups, d_tails, n_seg_total, n_groups, (int)seg_step, (int)n_avg, F, C, (float)(1.0 / (double)n_avg), d_psd);
  af_prof_end(ctx, AFRAME_PROF_WELCH, 2);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

// --------------------------------------------------------------------------------------------------
// The plain batched real transform of 8192 samples and its inverse (aframe_rfft8192 / aframe_irfft8192): the two halves
// of the whitening kernel without the spectral multiply, one work item per row.
//   rfft : x[8192] real -> X[0..4096] complex, X[k] = sum_n x[n] exp(-2 pi i n k / 8192)
//   irfft: X[0..4096] -> x[8192] real, with the 1/8192 (Im X[0], Im X[4096] are ignored)
// --------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(W64_THREADS, 2)
rfft8192_kernel(const float* __restrict__ x_in, int64_t n_items, const float2* __restrict__ tw, float2* __restrict__ spec) {
  constexpr int M = W64_M;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tab = reinterpret_cast<float2*>(smem_raw);
  const int tid = threadIdx.x, g = tid >> 6, t = tid & 63;
  float2* tile = tab + 4096 + g * F64_TILE;
  f64_fill_tab(tab, tw, tid, W64_THREADS);
  __syncthreads();
  const int bar = 1 + g;
  const float2 wt = __ldg(tw + t);               // W_8192^t
  for (int64_t item = (int64_t)blockIdx.x * 2 + g; item < n_items; item += (int64_t)gridDim.x * 2) {
    const float2* x2 = reinterpret_cast<const float2*>(x_in + item * AF_NOS);
    float2* X = spec + item * (M + 1);
    float2 v[64];
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      if (pass == 0) {
#pragma unroll
        for (int b = 0; b < 8; ++b)
#pragma unroll
          for (int a = 0; a < 8; ++a) v[8 * a + b] = __ldg(x2 + 64 * (8 * a + b) + t);
      } else {
        f64_load_row(v, tile, t);
      }
      fft64<-1>(v);
      if (pass == 0) { f64_twiddle_store<-1>(v, tile, tab, t); f64_bar(bar); }
    }
    mirror_publish(v, tile, t, bar);
#pragma unroll
    for (int k2 = 0; k2 < 32; ++k2) {
      const int k = t + 64 * k2;
      const float2 w = f64_cmul_cs<-1>(wt, w128_cs(k2));
      const float2 zk = v[k2], zq = *mirror_slot(tile, t, k2);
      const float2 ee = make_float2(zk.x + zq.x, zk.y - zq.y);          // 2 E
      const float2 oo = make_float2(zk.y + zq.y, zq.x - zk.x);          // 2 O
      const float2 wo = f64_cmul<false>(oo, w);
      X[k] = make_float2(0.5f * (ee.x + wo.x), 0.5f * (ee.y + wo.y));              // X[k] = E + W^k O
      X[M - k] = make_float2(0.5f * (ee.x - wo.x), -0.5f * (ee.y - wo.y));         // X[M - k] = conj(E - W^k O)
    }
    if (t == 0) X[M / 2] = make_float2(v[32].x, -v[32].y);                         // its own mirror: conj(Z[M/2])
    f64_bar(bar);
  }
}

__global__ void __launch_bounds__(W64_THREADS, 2)
irfft8192_kernel(const float2* __restrict__ spec, int64_t n_items, const float2* __restrict__ tw, float* __restrict__ x_out) {
  constexpr int M = W64_M;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* tab = reinterpret_cast<float2*>(smem_raw);
  const int tid = threadIdx.x, g = tid >> 6, t = tid & 63;
  float2* tile = tab + 4096 + g * F64_TILE;
  f64_fill_tab(tab, tw, tid, W64_THREADS);
  __syncthreads();
  const int bar = 1 + g;
  const float2 wt = __ldg(tw + t);
  const float sc = 0.5f / M;                     // the pair's half and the 1/M of the inverse
  for (int64_t item = (int64_t)blockIdx.x * 2 + g; item < n_items; item += (int64_t)gridDim.x * 2) {
    const float2* X = spec + item * (M + 1);
    float2 v[64];
    // pack: Z'[k] = X_E[k] + i X_O[k], kept conjugated for the forward code (IFFT(y) = conj(FFT(conj(y))))
#pragma unroll
    for (int k2 = 0; k2 < 32; ++k2) {
      const int k = t + 64 * k2;
      const float2 w = f64_cmul_cs<-1>(wt, w128_cs(k2));
      float2 yk = __ldg(X + k), ym = __ldg(X + M - k);
      if (k == 0) { yk.y = 0.f; ym.y = 0.f; }
      ym.y = -ym.y;                              // conj(X[M - k])
      const float2 ep = make_float2(sc * (yk.x + ym.x), sc * (yk.y + ym.y));
      const float2 op = f64_cmul<true>(make_float2(sc * (yk.x - ym.x), sc * (yk.y - ym.y)), w);
      v[k2] = make_float2(ep.x - op.y, -(ep.y + op.x));
      *mirror_slot(tile, t, k2) = make_float2(ep.x + op.y, ep.y - op.x);
    }
    if (t == 0) { const float2 xm = __ldg(X + M / 2); tile[32] = make_float2(xm.x * (1.0f / M), xm.y * (1.0f / M)); }
    f64_bar(bar);
#pragma unroll
    for (int k2 = 32; k2 < 64; ++k2) v[k2] = tile[t * F64_ROW + k2];
    f64_bar(bar);
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      if (pass == 1) f64_load_row(v, tile, t);
      fft64<-1>(v);
      if (pass == 0) { f64_twiddle_store<-1>(v, tile, tab, t); f64_bar(bar); }
    }
    float2* o = reinterpret_cast<float2*>(x_out + item * AF_NOS);
#pragma unroll
    for (int n1 = 0; n1 < 64; ++n1) o[64 * n1 + t] = make_float2(v[n1].x, -v[n1].y);
    f64_bar(bar);
  }
}

static std::atomic<uint64_t> g_rfft_attr{0}, g_irfft_attr{0};

AF_API aframe_status aframe_rfft8192(aframe_ctx* ctx, const float* d_x, int64_t batch, float* d_spec) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_x || !d_spec) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (batch < 0) return af_fail(ctx, AFRAME_EINVAL, "negative batch");
  if (batch == 0) return AFRAME_OK;
  if ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_spec)) & 7) return af_fail(ctx, AFRAME_EINVAL, "rfft8192: pointers must be 8-byte aligned");
  aframe_status st = w64_set_smem(ctx, rfft8192_kernel, g_rfft_attr);
  if (st != AFRAME_OK) return st;
  const int64_t want = (batch + 1) / 2, cap = 2 * (int64_t)ctx->n_sms;
  rfft8192_kernel<<<(unsigned)(want < cap ? want : cap), W64_THREADS, W64_SMEM, ctx->stream>>>(d_x, batch, ctx->d_tw32,
                                                                                             reinterpret_cast<float2*>(d_spec));
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}

AF_API aframe_status aframe_irfft8192(aframe_ctx* ctx, const float* d_spec, int64_t batch, float* d_x) {
  if (!ctx) return AFRAME_EINVAL;
  if (!d_x || !d_spec) return af_fail(ctx, AFRAME_EINVAL, "null pointer");
  if (batch < 0) return af_fail(ctx, AFRAME_EINVAL, "negative batch");
  if (batch == 0) return AFRAME_OK;
  if ((reinterpret_cast<uintptr_t>(d_x) | reinterpret_cast<uintptr_t>(d_spec)) & 7) return af_fail(ctx, AFRAME_EINVAL, "irfft8192: pointers must be 8-byte aligned");
  aframe_status st = w64_set_smem(ctx, irfft8192_kernel, g_irfft_attr);
  if (st != AFRAME_OK) return st;
  const int64_t want = (batch + 1) / 2, cap = 2 * (int64_t)ctx->n_sms;
  irfft8192_kernel<<<(unsigned)(want < cap ? want : cap), W64_THREADS, W64_SMEM, ctx->stream>>>(reinterpret_cast<const float2*>(d_spec),
                                                                                              batch, ctx->d_tw32, d_x);
  AF_LAUNCH_CHECK(ctx);
  return AFRAME_OK;
}
