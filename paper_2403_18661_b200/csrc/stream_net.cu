// O-6 streaming state, network part: the config-1 network of ONE window per update, computed incrementally.
//
// P:41 "snapshotting": consecutive 1.5 s windows overlap by all but `stride` samples, and (shared
// stages; the identity is pinned on the oracle alone in tests/test_oracle_network.py) a row of a layer's output is the
// same in every window that holds it unless it lies within reach of THAT window's zero padding: the first e and the last f
// rows of the layer's T rows.  The batched path uses this across the windows of a chunk; here it is used across UPDATES.
// Per layer the state keeps a ring of "stream" rows (the values a row has when real data surrounds it).  One update
// computes, per layer,
//     nnew = stride / (samples per row)   new stream rows   (window rows [T - f - nnew, T - f)),
//     e head rows (window rows [0, e), zero padding on the left) and f tail rows ([T - f, T), zero padding on the right),
// i.e. M = nnew + e + f <= 48 rows instead of T = 768 ... 96, reading every input row either from the input layer's ring
// or from its head / tail rows of this update.  e and f follow from the conv definition: an output row is an edge row iff
// one of the input rows it reads is padding or an edge row of the input (af_stream_net_plan_rows).
//
// One update = ONE kernel: a single thread-block cluster of CL CTAs (16 if the device can place one, else 8) x 512 threads
// walks the 37 layers; a layer is a [48 x K] x [K x C_out] product on mma.sync.m16n8k16 (fp16 in, fp32 accumulate -- the
// roundings of the batched tcgen05 path: fp16 weights, one fp16 rounding per stored activation; a 48-row product is far
// below the 128-row tcgen05 tile).  CTA c owns the 8-channel output blocks nb = c, c + CL, ...; its 16 warps split
// (block, K chunk), each warp streaming its B fragments from a fragment-ordered copy of the weights (one 16-byte cp.async
// per lane and two K steps, issued before the previous layer's cluster barrier) and reading A fragments with ldmatrix from
// a padded shared-memory copy of the layer's <= 56 input rows; partial sums meet in shared memory and the epilogue (+ bias,
// + residual, fp16, ReLU) stores rows to the ring / head / tail buffers in global memory (L2).  Layers are separated by one
// cluster barrier (release / acquire), not by kernel boundaries: 37 barriers of ~0.6 us replace ~36 launches of 5-7 us.
#include <cuda_runtime.h>
#include <new>
#include "common.cuh"
#include "stream_net.h"

namespace {

constexpr int SN_THREADS = 512;
constexpr int SN_WARPS = SN_THREADS / 32;
constexpr int SN_MAX_MT = 3;                      // 16-row tiles per layer (M <= 48)
constexpr int SN_MAX_LAYERS = 64;
constexpr int SN_PD = 12;                         // weight-fragment copies (pairs of K steps) a warp keeps in flight
constexpr int SN_PART_BYTES = SN_WARPS * SN_MAX_MT * 128 * 4;    // partial sums of the 16 warps
constexpr int SN_WBUF_BYTES = SN_WARPS * SN_PD * 512;            // weight fragments in flight
constexpr int SN_RES_BYTES = SN_THREADS * 16;                    // one residual piece per epilogue thread
constexpr int SN_BIAS_BYTES = SN_WARPS * 8 * 4;                  // the folded bias of this CTA's output blocks
constexpr int SN_GP = 8;                          // 16-byte pieces of the input rows per thread

struct SnLayer {
  int kind;                   // 0: conv on the tensor cores; 1: fused stem (conv + ReLU + max-pool k3 s2 p1) on CUDA cores
  int c_in, c_out, taps, P, pad, relu;
  int in_layer, res_layer;    // indices into the plan's layer array, -1 = none (stem: input = the whitened window)
  int T_in, T_out;            // rows of the input / output per window
  int e, f, nnew;             // head rows, tail rows, new stream rows per update
  int ring_mask;              // ring rows - 1 (power of two >= T_out)
  int m_rows;                 // nnew + e + f
  int seg_in_base[3];         // shared-memory row of the first input row of the stream / head / tail segment
  int in_rows;                // shared-memory input rows in total
  int kpt;                    // K steps (16 channels) per tap = c_in / 16
  int kpairs;                 // pairs of K steps = taps * c_in / 32
  int kc, ppc;                // K chunks per output block and pairs per chunk
  int is_last;                // feeds the head: the epilogue also emits per-row dot products with the head weights
  int conv_T, conv_P, conv_pad;   // stem only: rows / stride / padding of the conv before the pool
  long long ring_off, head_off, tail_off;   // element offsets into the activation arena
  long long w_off;            // uint4 offset into the fragment-ordered weights
  const float* bias;          // [c_out] folded bias (fp32)
  const float* w32;           // stem only: [taps][c_in][c_out] fp32
};

struct SnParams {
  const SnLayer* layers;
  int n_layers;
  __half* arena;
  const uint4* wfrag;
  const float* white;         // [C][K] fp32: the window (oldest sample first)
  int K;
  const int64_t* d_n;         // [0] raw samples received (the absolute clock of the rings)
  const int* d_has_filter;
  const int32_t* d_n_scores;  // written by the slide kernel of this update: 1 = the window is full
  int stride;
  float* head_part;           // [48][c_out / 8] per-row partial dot products of this update
  float* dr_ring;             // [ring rows of the last layer] per-row dot products of the stream rows
  const float* head_w;
  float head_b;
  float* d_scores;
};

__device__ __forceinline__ uint32_t sn_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t sn_cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t sn_cluster_size() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void sn_cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void sn_cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void sn_cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void sn_ldmatrix_x4(uint32_t addr, uint32_t (&a)[4]) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];"
               : "=r"(a[0]), "=r"(a[1]), "=r"(a[2]), "=r"(a[3]) : "r"(addr));
}
__device__ __forceinline__ void sn_mma(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 sn_ldcg(const uint4* p) { return __ldcg(p); }
__device__ __forceinline__ void sn_cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void sn_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void sn_cp_async_wait_1() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ void sn_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// window row r of layer L's output at the update whose ring base is `base` (= update index * nnew)
__device__ __forceinline__ const __half* sn_row(const SnLayer& L, const __half* arena, int r, long long base) {
  if (r < L.e) return arena + L.head_off + (long long)r * L.c_out;
  if (r >= L.T_out - L.f) return arena + L.tail_off + (long long)(r - (L.T_out - L.f)) * L.c_out;
  return arena + L.ring_off + (long long)((base + r) & L.ring_mask) * L.c_out;
}
// output row m of this update -> window row
__device__ __forceinline__ int sn_out_row(const SnLayer& L, int m) {
  if (m < L.nnew) return L.T_out - L.f - L.nnew + m;
  if (m < L.nnew + L.e) return m - L.nnew;
  return L.T_out - L.f + (m - L.nnew - L.e);
}
// shared-memory input row read by output row m for tap 0
__device__ __forceinline__ int sn_in_row0(const SnLayer& L, int m) {
  if (m < L.nnew) return L.seg_in_base[0] + L.P * m;
  if (m < L.nnew + L.e) return L.seg_in_base[1] + L.P * (m - L.nnew);
  return L.seg_in_base[2] + L.P * (m - L.nnew - L.e);
}
// work item of a warp in layer L: output block nb = rank + (warp / kc) CL, pairs [pair0, pair0 + npairs) of its K steps
__device__ __forceinline__ void sn_item(const SnLayer& L, int rank, int CL, int warp, int lane, const uint4* wfrag, int& npairs,
                                        const uint4*& wp) {
  const int NB = L.c_out >> 3;
  const int nbl = (NB - rank + CL - 1) / CL;
  const int bi = warp / L.kc, kci = warp - bi * L.kc;
  const int nb = rank + bi * CL;
  const int pair0 = kci * L.ppc;
  npairs = L.kpairs - pair0;
  if (npairs > L.ppc) npairs = L.ppc;
  if (bi >= nbl || npairs < 0) npairs = 0;
  wp = wfrag + L.w_off + ((long long)nb * L.kpairs + pair0) * 32 + lane;
}

#ifdef AFRAME_TC_CYCLES   // experiments build only: phase times (ns, globaltimer) of CTA 0, thread 0: [layer][5]
__device__ unsigned long long g_sn_times[SN_MAX_LAYERS * 5 + 8];
#define SN_T(li, k) do { if (tid == 0 && rank == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_sn_times[(li) * 5 + (k)] = t_; } } while (0)
#else
#define SN_T(li, k) do { } while (0)
#endif

__global__ void __launch_bounds__(SN_THREADS, 1) stream_net_kernel(const SnParams p) {
  extern __shared__ __align__(16) unsigned char sn_smem[];
  if (*p.d_has_filter == 0) return;                // no whitened sample yet (uniform over the cluster)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int rank = (int)sn_cluster_rank(), CL = (int)sn_cluster_size();
  const long long upd = p.d_n[0] / p.stride;       // absolute update index: the rings' clock
  __shared__ SnLayer s_layers[SN_MAX_LAYERS];      // the plan
  for (int i = tid; i < p.n_layers * (int)(sizeof(SnLayer) / 4); i += SN_THREADS)
    reinterpret_cast<uint32_t*>(s_layers)[i] = reinterpret_cast<const uint32_t*>(p.layers)[i];
  __syncthreads();
  // dynamic shared memory: partial sums of the 16 warps | weight fragments in flight | residual pieces | the layer's input rows
  float* part = reinterpret_cast<float*>(sn_smem);
  // this warp's weight fragments in flight: SN_PD pairs of K steps, one 16-byte cp.async per lane and pair (asynchronous
  // copies cannot be sunk to their first use by the compiler, which is what happened to plain loads held in registers)
  uint4* wbuf = reinterpret_cast<uint4*>(sn_smem + SN_PART_BYTES) + warp * (SN_PD * 32) + lane;
  uint4* res_buf = reinterpret_cast<uint4*>(sn_smem + SN_PART_BYTES + SN_WBUF_BYTES);
  float* bias_buf = reinterpret_cast<float*>(sn_smem + SN_PART_BYTES + SN_WBUF_BYTES + SN_RES_BYTES);
  unsigned char* in_tile = sn_smem + SN_PART_BYTES + SN_WBUF_BYTES + SN_RES_BYTES + SN_BIAS_BYTES;
  auto sn_prefetch = [&](int li) {
    if (li >= p.n_layers || s_layers[li].kind != 0) { sn_cp_async_commit(); return; }   // (an empty group: the epilogue counts groups)
    int np;
    const uint4* w;
    sn_item(s_layers[li], rank, CL, warp, lane, p.wfrag, np, w);
#pragma unroll
    for (int j = 0; j < SN_PD; ++j)
      if (j < np) sn_cp_async16(sn_smem_u32(wbuf + j * 32), w + j * 32);
    sn_cp_async_commit();
  };
  sn_prefetch(1);                                  // (layer 0 is the stem)

  for (int li = 0; li < p.n_layers; ++li) {
    const SnLayer& L = s_layers[li];
    const long long base = upd * L.nnew;
    SN_T(li, 0);
    if (L.kind == 1) {
      // ---- fused stem: conv (k7 s2) + bias + ReLU + max-pool k3 s2 p1 from the fp32 window, same FMA order as stem_pool_kernel
      const int n_items = L.m_rows * L.c_out;
      for (int it = rank * SN_THREADS + tid; it < n_items; it += CL * SN_THREADS) {
        const int m = it / L.c_out, co = it - m * L.c_out;
        const int r = sn_out_row(L, m);
        const bool padded = m >= L.nnew;           // head / tail rows see the window's zero padding; stream rows never reach it
        // k7 s2 p3 on two channels (af_stream_net_create checks it): conv positions 2r-1, 2r, 2r+1 read samples 4r-5 .. 4r+5.
        // All loads first (one round trip), then the FMAs in stem_pool_kernel's order (bias; channel outer, tap inner).
        float x[2][11], wv[7][2];
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
          for (int i = 0; i < 11; ++i) {
            const int s = 4 * r - 5 + i;
            x[c][i] = (!padded || (s >= 0 && s < p.K)) ? p.white[(long long)c * p.K + s] : 0.f;
          }
#pragma unroll
        for (int d = 0; d < 7; ++d)
#pragma unroll
          for (int c = 0; c < 2; ++c) wv[d][c] = __ldg(L.w32 + (d * 2 + c) * L.c_out + co);
        const float bs = __ldg(L.bias + co);
        float best = 0.f;                          // (ReLU output >= 0: a missing pool position never wins)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const int t = 2 * r - 1 + j;
          float acc = bs;
#pragma unroll
          for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int d = 0; d < 7; ++d) acc = fmaf(wv[d][c], x[c][2 * j + d], acc);
          if (t >= 0 && t < L.conv_T) best = fmaxf(best, fmaxf(acc, 0.f));
        }
        __half* dst = const_cast<__half*>(sn_row(L, p.arena, r, base)) + co;
        if (m < L.nnew) dst = p.arena + L.ring_off + (long long)((base + r) & L.ring_mask) * L.c_out + co;
        *dst = __float2half_rn(fminf(best, 65504.f));
      }
      SN_T(li, 3);
      sn_cluster_sync();
      SN_T(li, 4);
      continue;
    }
    // ---- conv layer on the tensor cores
    const SnLayer& Lin = s_layers[L.in_layer];
    const long long base_in = upd * Lin.nnew;
    const int NB = L.c_out >> 3;
    const int nbl = (NB - rank + CL - 1) / CL;     // output blocks of this CTA: nb = rank + i CL
    // this warp's work item (block i, K chunk k) = (warp / kc, warp % kc); its first weight fragments are already in flight:
    // they do not depend on the activations and were issued before the previous layer's barrier (sn_prefetch)
    int npairs;
    const uint4* wp;
    sn_item(L, rank, CL, warp, lane, p.wfrag, npairs, wp);

    // the residual piece this thread's epilogue item adds travels meanwhile (item = tid; items past 512 load theirs directly)
    const int n_epi = L.m_rows * nbl;
    if (L.res_layer >= 0 && tid < n_epi) {
      const int m = tid / nbl, i = tid - m * nbl;
      const SnLayer& Lr = s_layers[L.res_layer];
      sn_cp_async16(sn_smem_u32(res_buf + tid),
                    reinterpret_cast<const uint4*>(sn_row(Lr, p.arena, sn_out_row(L, m), upd * Lr.nnew)) + (rank + i * CL));
    }
    if (tid < 2 * nbl)                             // ... and the bias of this CTA's blocks (block i = tid / 2: channels 8 (rank + i CL) ...)
      sn_cp_async16(sn_smem_u32(bias_buf + 4 * tid), L.bias + (rank + (tid >> 1) * CL) * 8 + 4 * (tid & 1));
    sn_cp_async_commit();

    // gather the input rows (16-byte pieces; rows padded by 16 B: conflict-free ldmatrix)
    const int row_bytes = L.c_in * 2 + 16;
    {
      const int ppr_log = 31 - __clz(L.c_in >> 3);  // pieces per row (c_in / 8, a power of two)
      const int total = L.in_rows << ppr_log;
      // asynchronous copies straight into shared memory (<= SN_GP pieces per thread, all in flight at once); rows outside the
      // window are written as zeros.  (One bulk copy per row instead was measured: 2.3-2.9 us per layer against 0.9-2.2.)
#pragma unroll
      for (int k = 0; k < SN_GP; ++k) {
        const int i = tid + k * SN_THREADS;
        if (i < total) {
          const int j = i >> ppr_log, q = i - (j << ppr_log);
          const int s = j >= L.seg_in_base[2] ? 2 : (j >= L.seg_in_base[1] ? 1 : 0);
          const int r_first = s == 0 ? L.T_out - L.f - L.nnew : (s == 1 ? 0 : L.T_out - L.f);
          const int r_in = L.P * r_first - L.pad + (j - L.seg_in_base[s]);
          unsigned char* dst = in_tile + (size_t)j * row_bytes + q * 16;
          if (r_in >= 0 && r_in < L.T_in) sn_cp_async16(sn_smem_u32(dst), reinterpret_cast<const uint4*>(sn_row(Lin, p.arena, r_in, base_in)) + q);
          else *reinterpret_cast<uint4*>(dst) = make_uint4(0, 0, 0, 0);
        }
      }
      sn_cp_async_commit();
      sn_cp_async_wait_all();
    }
    __syncthreads();
    SN_T(li, 1);

    // main loop: acc[mt] += A[mt](16 x 16) B(16 x 8) over this warp's K chunk
    float acc[SN_MAX_MT][4];
#pragma unroll
    for (int mt = 0; mt < SN_MAX_MT; ++mt) { acc[mt][0] = acc[mt][1] = acc[mt][2] = acc[mt][3] = 0.f; }
    if (npairs > 0) {
      const int n_mt = (L.m_rows + 15) >> 4;
      uint32_t a_base[SN_MAX_MT];
#pragma unroll
      for (int mt = 0; mt < SN_MAX_MT; ++mt) {
        int m = mt * 16 + (lane & 7) + ((lane >> 3) & 1) * 8;
        if (m >= L.m_rows) m = 0;                  // rows past M read row 0 (their results are dropped)
        a_base[mt] = sn_smem_u32(in_tile) + (uint32_t)(sn_in_row0(L, m) * row_bytes + (lane >> 4) * 16);
      }
      int ks = 2 * ((warp % L.kc) * L.ppc);
      int d = ks / L.kpt, kcol = ks - d * L.kpt;   // tap and 16-channel step of K step ks
      for (int pi0 = 0; pi0 < npairs; pi0 += SN_PD) {
        sn_cp_async_wait_all();                    // (each lane reads back only what it copied itself)
#pragma unroll
        for (int j = 0; j < SN_PD; ++j) {
          if (pi0 + j < npairs) {
            const uint4 bq = wbuf[j * 32];
            const uint32_t bb[4] = {bq.x, bq.y, bq.z, bq.w};
            if (pi0 + j + SN_PD < npairs) sn_cp_async16(sn_smem_u32(wbuf + j * 32), wp + (pi0 + j + SN_PD) * 32);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const uint32_t off = (uint32_t)(d * row_bytes + kcol * 32);
#pragma unroll
              for (int mt = 0; mt < SN_MAX_MT; ++mt) {
                if (mt < n_mt) {
                  uint32_t a[4];
                  sn_ldmatrix_x4(a_base[mt] + off, a);
                  sn_mma(acc[mt], a, bb[2 * h], bb[2 * h + 1]);
                }
              }
              if (++kcol == L.kpt) { kcol = 0; ++d; }
            }
          }
        }
        sn_cp_async_commit();                      // (the refills of this round, if any)
      }
    }
    // partial sums -> shared memory: part[warp][mt][reg][lane]
#pragma unroll
    for (int mt = 0; mt < SN_MAX_MT; ++mt)
#pragma unroll
      for (int j = 0; j < 4; ++j) part[((warp * SN_MAX_MT + mt) * 4 + j) * 32 + lane] = acc[mt][j];
    sn_cp_async_wait_all();                        // this thread's residual / bias pieces have landed; after the barrier everyone's
    __syncthreads();
    SN_T(li, 2);

    // epilogue: one thread per (output row, output block): sum the K chunks in order, + bias (+ residual) -> fp16 -> ReLU
    {
      for (int it = tid; it < n_epi; it += SN_THREADS) {
        const int m = it / nbl, i = it - m * nbl;
        const int nbo = rank + i * CL;
        const int mt = m >> 4, rr = m & 15;
        float v[8];
        {
          const float4 b0 = reinterpret_cast<const float4*>(bias_buf)[2 * i], b1 = reinterpret_cast<const float4*>(bias_buf)[2 * i + 1];
          v[0] = b0.x; v[1] = b0.y; v[2] = b0.z; v[3] = b0.w; v[4] = b1.x; v[5] = b1.y; v[6] = b1.z; v[7] = b1.w;
        }
        // accumulator fragment of m16n8: lane = (row % 8) * 4 + col / 2, register = (row / 8) * 2 + col % 2
        for (int k = 0; k < L.kc; ++k) {
          const int w = i * L.kc + k;
          // (the row's even columns are register (rr / 8) * 2 of four consecutive lanes, its odd columns the next register)
          const float* pp = part + (size_t)(w * SN_MAX_MT + mt) * 128 + (rr >> 3) * 64 + (rr & 7) * 4;
          const float4 ev = *reinterpret_cast<const float4*>(pp), od = *reinterpret_cast<const float4*>(pp + 32);
          v[0] += ev.x; v[1] += od.x; v[2] += ev.y; v[3] += od.y; v[4] += ev.z; v[5] += od.z; v[6] += ev.w; v[7] += od.w;
        }
        const int r = sn_out_row(L, m);
        if (L.res_layer >= 0) {
          const SnLayer& Lr = s_layers[L.res_layer];
          const uint4 rv = it < SN_THREADS ? res_buf[it] : sn_ldcg(reinterpret_cast<const uint4*>(sn_row(Lr, p.arena, r, upd * Lr.nnew)) + nbo);
          const uint32_t rw[4] = {rv.x, rv.y, rv.z, rv.w};
#pragma unroll
          for (int q = 0; q < 4; ++q) { const float2 t = af_act_unpack2(rw[q]); v[2 * q] += t.x; v[2 * q + 1] += t.y; }
        }
        uint32_t ow[4];
        const __half2 lo2 = __float2half2_rn(L.relu ? 0.f : -INFINITY);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const uint32_t pk = af_act_pack2(v[2 * q], v[2 * q + 1]);
          const __half2 mx = __hmax2(*reinterpret_cast<const __half2*>(&pk), lo2);
          ow[q] = *reinterpret_cast<const uint32_t*>(&mx);
        }
        __half* dst;
        if (m < L.nnew) dst = p.arena + L.ring_off + (long long)((base + r) & L.ring_mask) * L.c_out;
        else if (m < L.nnew + L.e) dst = p.arena + L.head_off + (long long)r * L.c_out;
        else dst = p.arena + L.tail_off + (long long)(r - (L.T_out - L.f)) * L.c_out;
        *reinterpret_cast<uint4*>(dst + nbo * 8) = make_uint4(ow[0], ow[1], ow[2], ow[3]);
        if (L.is_last) {                           // the head's dot product of this row over these 8 channels
          float s = 0.f;
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const float2 t = af_act_unpack2(ow[q]);
            s = fmaf(t.x, p.head_w[nbo * 8 + 2 * q], s);
            s = fmaf(t.y, p.head_w[nbo * 8 + 2 * q + 1], s);
          }
          p.head_part[m * NB + nbo] = s;
        }
      }
    }
    SN_T(li, 3);
    // this layer's rows become visible to every CTA; the next layer's first weight fragments (which depend on no activation)
    // are issued between the arrival and the wait, so that their issue time hides in the barrier's latency
    sn_cluster_arrive();
    sn_prefetch(li + 1);
    sn_cluster_wait();
    SN_T(li, 4);
  }

  // ---- head: global average pool + linear (reading B8) from per-row dot products
  if (rank == 0) {
    const SnLayer& L = s_layers[p.n_layers - 1];
    const long long base = upd * L.nnew;
    const int NB = L.c_out >> 3;
    float* rowdot = part;                          // [T_out]
    for (int m = tid; m < L.m_rows; m += SN_THREADS) {
      float s = 0.f;
      for (int b = 0; b < NB; ++b) s += __ldcg(p.head_part + m * NB + b);
      const int r = sn_out_row(L, m);
      rowdot[r] = s;
      if (m < L.nnew) p.dr_ring[(base + r) & L.ring_mask] = s;
    }
    __syncthreads();
    for (int r = L.e + tid; r < L.T_out - L.f - L.nnew; r += SN_THREADS) rowdot[r] = __ldcg(p.dr_ring + ((base + r) & L.ring_mask));
    __syncthreads();
    if (warp == 0) {                               // fixed order: lane l sums rows l, l + 32, ...; then a shuffle tree
      float s = 0.f;
      for (int r = lane; r < L.T_out; r += 32) s += rowdot[r];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane == 0 && *p.d_n_scores == 1) p.d_scores[0] = s / (float)L.T_out + p.head_b;
    }
    SN_T(SN_MAX_LAYERS, 0);
  }
}

// fragment-ordered copy of a conv layer's fp16 weights W[tap][c_out][c_in]:
// out[((nb * kpairs + pair) * 32 + lane) * 4 + j]: K step ks = 2 pair + j / 2, tap d = ks / (c_in / 16), ci0 = 16 (ks % (c_in / 16)),
// register j % 2 of the m16n8k16 B fragment = W[d][8 nb + lane / 4][ci0 + 8 (j % 2) + 2 (lane % 4) + {0, 1}]
__global__ void sn_pack_weights_kernel(const __half* __restrict__ w, int c_in, int c_out, int taps, uint32_t* __restrict__ out) {
  const int kpt = c_in / 16, kpairs = taps * c_in / 32;
  const long long total = (long long)(c_out / 8) * kpairs * 128;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(i & 3), lane = (int)((i >> 2) & 31);
    const long long pr = i >> 7;
    const int pair = (int)(pr % kpairs), nb = (int)(pr / kpairs);
    const int ks = 2 * pair + (j >> 1), d = ks / kpt, ci0 = 16 * (ks % kpt);
    const int co = 8 * nb + (lane >> 2), ci = ci0 + 8 * (j & 1) + 2 * (lane & 3);
    const __half* src = w + ((long long)d * c_out + co) * c_in + ci;
    out[i] = (uint32_t)__half_as_ushort(src[0]) | ((uint32_t)__half_as_ushort(src[1]) << 16);
  }
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------------

struct af_stream_net {
  std::vector<SnLayer> layers;
  SnLayer* d_layers = nullptr;
  __half* d_arena = nullptr;
  size_t arena_bytes = 0;
  uint4* d_wfrag = nullptr;
  float* d_head_part = nullptr;
  float* d_dr_ring = nullptr;
  size_t dr_bytes = 0;
  int cluster = 0;
  int smem_bytes = 0;
  const float* d_head_w = nullptr;
  float head_b = 0.f;
};

// Edge rows of a layer's output from those of its input (see the file header): output row t reads input rows
// P t - pad ... P t - pad + k - 1; it is a head row iff P t - pad < e_in, a tail row iff P t - pad + k - 1 >= T_in - f_in.
static void sn_edges(int T_in, int e_in, int f_in, int k, int P, int pad, int T_out, int& e, int& f) {
  e = (e_in + pad + P - 1) / P;
  int t_star = T_in - f_in - k + 1 + pad;          // first t with P t >= t_star is a tail row
  t_star = t_star <= 0 ? 0 : (t_star + P - 1) / P;
  f = T_out - t_star;
  if (e > T_out) e = T_out;
  if (f < 0) f = 0;
}

bool af_stream_net_plan_rows(const std::vector<LayerDesc>& table, int stride, std::vector<int>* e_out, std::vector<int>* f_out,
                             std::vector<int>* new_out, const char** why) {
  static const char* ok = "";
  *why = ok;
  const int n = (int)table.size();
  if (n < 4 || table[0].kind != 0 || table[1].kind != 1 || table[n - 1].kind != 2) { *why = "layer pattern is not stem conv, pool, convs, head"; return false; }
  if (table[1].k != 3 || table[1].stride != 2 || table[1].pad != 1 || table[1].input_from != 0 || !table[0].relu) { *why = "stem pool is not k3 s2 p1 after a ReLU"; return false; }
  std::vector<int> e(n, 0), f(n, 0), D(n, 1), nw(n, 0);
  for (int i = 0; i < n - 1; ++i) {
    const LayerDesc& l = table[i];
    if (i >= 2 && (l.kind != 0 || l.input_from < 1)) { *why = "layer pattern is not stem conv, pool, convs, head"; return false; }
    const int src = l.input_from;
    const int e_in = src < 0 ? 0 : e[src], f_in = src < 0 ? 0 : f[src], d_in = src < 0 ? 1 : D[src];
    sn_edges(l.t_in, e_in, f_in, l.k, l.stride, l.pad, l.t_out, e[i], f[i]);
    D[i] = d_in * l.stride;
    if (stride % D[i]) { *why = "stride is not a multiple of the network's total downsampling"; return false; }
    nw[i] = stride / D[i];
    if (l.residual_from >= 0) {
      const int rs = l.residual_from;
      if (D[rs] != D[i] || e[rs] > e[i] || f[rs] > f[i]) { *why = "residual rows do not line up"; return false; }
    }
    if (i >= 1 && (e[i] + f[i] + nw[i] > 16 * SN_MAX_MT || e[i] + nw[i] + f[i] > l.t_out)) { *why = "more than 48 rows per layer and update"; return false; }
    if (i >= 2 && (l.c_in % 32 || l.c_out % 8 || (l.k != 1 && l.k != 3) || l.c_in > 512)) { *why = "channel counts the fragment layout cannot take"; return false; }
  }
  if (table[n - 1].input_from != n - 2) { *why = "head does not read the last conv"; return false; }
  if (e_out) *e_out = e;
  if (f_out) *f_out = f;
  if (new_out) *new_out = nw;
  return true;
}

void af_stream_net_free(af_stream_net* sn) {
  if (!sn) return;
  cudaFree(sn->d_layers); cudaFree(sn->d_arena); cudaFree(sn->d_wfrag); cudaFree(sn->d_head_part); cudaFree(sn->d_dr_ring);
  cudaGetLastError();
  delete sn;
}

aframe_status af_stream_net_reset(aframe_ctx* ctx, af_stream_net* sn) {
  AF_CUDA(ctx, cudaMemsetAsync(sn->d_arena, 0, sn->arena_bytes, ctx->stream));
  AF_CUDA(ctx, cudaMemsetAsync(sn->d_dr_ring, 0, sn->dr_bytes, ctx->stream));
  return AFRAME_OK;
}

static int sn_pow2_at_least(int v) { int p = 1; while (p < v) p <<= 1; return p; }

aframe_status af_stream_net_create(aframe_ctx* ctx, const aframe_weights* w, af_stream_net** out, const char** why) {
  *out = nullptr;
  static const char* ok = "";
  *why = ok;
  const aframe_config& cfg = ctx->cfg;
  if (cfg.precision != AFRAME_F16 || !w->tc_ok || w->live_gn) { *why = "not the folded tensor-core path"; return AFRAME_OK; }
  if (cfg.stride > 128) { *why = "stride above 128 samples"; return AFRAME_OK; }
  std::vector<int> e, f, nw;
  if (!af_stream_net_plan_rows(w->layers, cfg.stride, &e, &f, &nw, why)) return AFRAME_OK;
  const int n = (int)w->layers.size();
  if (n - 2 > SN_MAX_LAYERS) { *why = "too many layers"; return AFRAME_OK; }
  af_stream_net* sn = new (std::nothrow) af_stream_net();
  if (!sn) return af_fail(ctx, AFRAME_ENOMEM, "host allocation failed");
  int smem_in_max = 0;
  std::vector<int> map(n, -1);                     // layer table index -> plan index (the pool stands for the fused stem)
  long long arena = 0, wfrag = 0;
  for (int i = 1; i < n - 1; ++i) {
    const LayerDesc& l = w->layers[i];
    SnLayer L = {};
    map[i] = (int)sn->layers.size();
    L.kind = i == 1 ? 1 : 0;
    const LayerDesc& cv = i == 1 ? w->layers[0] : l;
    L.c_in = cv.c_in; L.c_out = l.c_out; L.taps = cv.k; L.P = l.stride; L.pad = l.pad; L.relu = l.relu;
    L.in_layer = i == 1 ? -1 : map[l.input_from];
    L.res_layer = l.residual_from >= 0 ? map[l.residual_from] : -1;
    L.T_in = l.t_in; L.T_out = l.t_out;
    L.e = e[i]; L.f = f[i]; L.nnew = nw[i];
    L.ring_mask = sn_pow2_at_least(l.t_out) - 1;
    L.m_rows = L.nnew + L.e + L.f;
    L.is_last = i == n - 2;
    L.bias = i == 1 ? w->d_bias[0] : w->d_bias[i];
    if (i == 1) {
      if (cv.k != 7 || cv.c_in != 2 || cv.stride != 2 || cv.pad != 3) { delete sn; *why = "stem conv is not k7 s2 p3 on two channels"; return AFRAME_OK; }
      L.conv_T = cv.t_out; L.conv_P = cv.stride; L.conv_pad = cv.pad;
      L.w32 = w->d_w32[0];
    } else {
      if (L.in_layer < 0 || (l.residual_from >= 0 && L.res_layer < 0)) { delete sn; *why = "layer reads the raw window or the stem conv"; return AFRAME_OK; }
      const int n_seg[3] = {L.nnew, L.e, L.f};
      int rows = 0;
      for (int s = 0; s < 3; ++s) { L.seg_in_base[s] = rows; rows += n_seg[s] > 0 ? L.P * (n_seg[s] - 1) + L.taps : 0; }
      L.in_rows = rows;
      if (rows * (L.c_in / 8) > SN_GP * SN_THREADS || (L.c_in & (L.c_in - 1))) { delete sn; *why = "input rows exceed the gather's capacity"; return AFRAME_OK; }
      const int bytes = rows * (L.c_in * 2 + 16);
      if (bytes > smem_in_max) smem_in_max = bytes;
      L.kpt = L.c_in / 16; L.kpairs = L.taps * L.c_in / 32;
      L.w_off = wfrag;
      wfrag += (long long)(L.c_out / 8) * L.kpairs * 32;
    }
    L.ring_off = arena; arena += (long long)(L.ring_mask + 1) * L.c_out;
    L.head_off = arena; arena += (long long)L.e * L.c_out;
    L.tail_off = arena; arena += (long long)L.f * L.c_out;
    arena = (arena + 63) & ~63ll;
    sn->layers.push_back(L);
  }
  sn->smem_bytes = SN_PART_BYTES + SN_WBUF_BYTES + SN_RES_BYTES + SN_BIAS_BYTES + smem_in_max;
  if (sn->smem_bytes > 200 * 1024) { delete sn; *why = "input rows do not fit shared memory"; return AFRAME_OK; }
  cudaError_t ce = cudaFuncSetAttribute(stream_net_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sn->smem_bytes);
  if (ce == cudaSuccess) ce = cudaFuncSetAttribute(stream_net_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  if (ce != cudaSuccess) { cudaGetLastError(); delete sn; return af_fail(ctx, AFRAME_ECUDA, "stream_net_kernel attributes: %s", cudaGetErrorString(ce)); }
  // cluster size: 16 CTAs if the device can place such a cluster, else 8
  sn->cluster = 8;
  {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(16); lc.blockDim = dim3(SN_THREADS); lc.dynamicSmemBytes = (size_t)sn->smem_bytes;
    cudaLaunchAttribute at;
    at.id = cudaLaunchAttributeClusterDimension;
    at.val.clusterDim.x = 16; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
    lc.attrs = &at; lc.numAttrs = 1;
    int n_cl = 0;
    if (cfg.stream_full_forward != 2 && cudaOccupancyMaxActiveClusters(&n_cl, stream_net_kernel, &lc) == cudaSuccess && n_cl >= 1) sn->cluster = 16;
    cudaGetLastError();
  }
  // work split per layer: the CTA with the most output blocks has nbl_max of them; its 16 warps take (block, K chunk)
  for (SnLayer& L : sn->layers) {
    if (L.kind != 0) continue;
    const int NB = L.c_out / 8;
    const int nbl_max = (NB + sn->cluster - 1) / sn->cluster;
    if (nbl_max > SN_WARPS) { af_stream_net_free(sn); *why = "more output blocks per CTA than warps"; return AFRAME_OK; }
    int kc = SN_WARPS / nbl_max;
    if (kc > L.kpairs) kc = L.kpairs;
    L.ppc = (L.kpairs + kc - 1) / kc;
    L.kc = (L.kpairs + L.ppc - 1) / L.ppc;
  }
  sn->arena_bytes = (size_t)arena * sizeof(__half);
  const SnLayer& last = sn->layers.back();
  sn->dr_bytes = (size_t)(last.ring_mask + 1) * sizeof(float);
  bool okm = cudaMalloc(&sn->d_layers, sn->layers.size() * sizeof(SnLayer)) == cudaSuccess &&
             cudaMalloc(&sn->d_arena, sn->arena_bytes) == cudaSuccess &&
             cudaMalloc(&sn->d_wfrag, (size_t)wfrag * sizeof(uint4)) == cudaSuccess &&
             cudaMalloc(&sn->d_head_part, (size_t)16 * SN_MAX_MT * (last.c_out / 8) * sizeof(float)) == cudaSuccess &&
             cudaMalloc(&sn->d_dr_ring, sn->dr_bytes) == cudaSuccess;
  if (!okm) { cudaGetLastError(); af_stream_net_free(sn); return af_fail(ctx, AFRAME_ENOMEM, "device allocation failed"); }
  if (cudaMemcpyAsync(sn->d_layers, sn->layers.data(), sn->layers.size() * sizeof(SnLayer), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess) {
    cudaGetLastError(); af_stream_net_free(sn); return af_fail(ctx, AFRAME_ECUDA, "plan upload failed");
  }
  for (int i = 2; i < n - 1; ++i) {
    const SnLayer& L = sn->layers[map[i]];
    sn_pack_weights_kernel<<<256, 256, 0, ctx->stream>>>(reinterpret_cast<const __half*>(w->d_w16[i]), L.c_in, L.c_out, L.taps,
                                                        reinterpret_cast<uint32_t*>(sn->d_wfrag + L.w_off));
  }
  if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(ctx->stream) != cudaSuccess) {
    cudaGetLastError(); af_stream_net_free(sn); return af_fail(ctx, AFRAME_ECUDA, "weight packing failed");
  }
  sn->d_head_w = w->d_head_w; sn->head_b = w->head_b;
  aframe_status rs = af_stream_net_reset(ctx, sn);
  if (rs != AFRAME_OK) { af_stream_net_free(sn); return rs; }
  *out = sn;
  return AFRAME_OK;
}

aframe_status af_stream_net_launch(aframe_ctx* ctx, af_stream_net* sn, const float* d_white, const int64_t* d_n,
                                   const int* d_has_filter, const int32_t* d_n_scores, float* d_scores) {
  SnParams p = {};
  p.layers = sn->d_layers; p.n_layers = (int)sn->layers.size();
  p.arena = sn->d_arena; p.wfrag = sn->d_wfrag; p.white = d_white; p.K = ctx->cfg.kernel_len;
  p.d_n = d_n; p.d_has_filter = d_has_filter; p.d_n_scores = d_n_scores; p.stride = ctx->cfg.stride;
  p.head_part = sn->d_head_part; p.dr_ring = sn->d_dr_ring; p.head_w = sn->d_head_w; p.head_b = sn->head_b;
  p.d_scores = d_scores;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)sn->cluster); lc.blockDim = dim3(SN_THREADS); lc.dynamicSmemBytes = (size_t)sn->smem_bytes;
  lc.stream = ctx->stream;
  cudaLaunchAttribute at;
  at.id = cudaLaunchAttributeClusterDimension;
  at.val.clusterDim.x = (unsigned)sn->cluster; at.val.clusterDim.y = 1; at.val.clusterDim.z = 1;
  lc.attrs = &at; lc.numAttrs = 1;
  af_prof_begin(ctx, AFRAME_PROF_STREAM);
  AF_CUDA(ctx, cudaLaunchKernelEx(&lc, stream_net_kernel, p));
  af_prof_end(ctx, AFRAME_PROF_STREAM, 1);
  ctx->launches++;
  return AFRAME_OK;
}

int af_stream_net_cluster(const af_stream_net* sn) { return sn ? sn->cluster : 0; }

#ifdef AFRAME_TC_CYCLES
AF_API int aframe_experiment_sn_times(unsigned long long* host_out /* [SN_MAX_LAYERS * 5 + 8] */) {
  cudaDeviceSynchronize();
  return (int)cudaMemcpyFromSymbol(host_out, g_sn_times, sizeof(unsigned long long) * (SN_MAX_LAYERS * 5 + 8));
}
#endif

aframe_status af_parse_layer_table(const void* host_blob, size_t bytes, int kernel_len, int n_channels,
                                   std::vector<LayerDesc>& layers, uint32_t hdr[8], const char** why);   // aframe_api.cu

// Host-only description of the incremental plan for a weight blob and an update stride (include/aframe.h).
AF_API aframe_status aframe_describe_stream_plan(const void* host_blob, size_t bytes, int32_t kernel_len, int32_t n_channels,
                                                 int32_t stride, int32_t max_layers, int32_t* n_layers, int32_t* t_out,
                                                 int32_t* head_rows, int32_t* tail_rows, int32_t* new_rows) {
  if (!host_blob || !n_layers || kernel_len < 1 || stride < 1 || max_layers < 0 ||
      (max_layers > 0 && (!t_out || !head_rows || !tail_rows || !new_rows))) return AFRAME_EINVAL;
  std::vector<LayerDesc> layers;
  uint32_t hdr[8];
  const char* why = "";
  const aframe_status st = af_parse_layer_table(host_blob, bytes, kernel_len, n_channels, layers, hdr, &why);
  if (st != AFRAME_OK) return st;
  *n_layers = 0;
  std::vector<int> e, f, nw;
  if (hdr[3] == 2 || stride > 128 || !af_stream_net_plan_rows(layers, stride, &e, &f, &nw, &why)) return AFRAME_OK;
  const int n = (int)layers.size() - 1;            // (the head holds no rows)
  *n_layers = n;
  for (int i = 0; i < n && i < max_layers; ++i) { t_out[i] = layers[i].t_out; head_rows[i] = e[i]; tail_rows[i] = f[i]; new_rows[i] = nw[i]; }
  return AFRAME_OK;
}
