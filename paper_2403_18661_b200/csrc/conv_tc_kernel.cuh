// 1D convolution (k = 1 or 3, stride 1 or 2) as an implicit GEMM on the 5th-gen tensor cores.
//
//   out[b][t][co] = relu( bias[co] + sum_{d, ci} W'[d][co][ci] * in[b][P*t + d - pad][ci] (+ res[b][t][co]) )
//
//   GEMM view: M = (window, t) rows, N = C_out, K = taps * C_in.  Activations are channels-last bf16, so a
//   row of A for tap d is the contiguous channel vector of input row P*t + d - pad.
//   A tile (128 rows x 64 ch) : ONE TMA box of the rank-4 view (C_in, P, T_in/P, B), start row shifted per
//                               tap; out-of-range rows (t = -1, T) are zero-filled by TMA = 'same' padding,
//                               per window, so rows never bleed between windows.  Stride 2 = parity dim.
//   B tile (BN x 64 ch)       : TMA box of the folded bf16 weights [taps][C_out][C_in] (K-major).
//   tcgen05.mma M=128, N=BN, K=16, fp32 accumulators in TMEM (two stages of BN columns).
//   Epilogue: tcgen05.ld -> +bias (+residual via TMA) -> ReLU -> bf16 -> swizzled smem -> TMA store.
//
// Warp roles (192 threads): warp 0 TMA producer, warp 1 MMA issuer (+TMEM alloc), warps 2-5 epilogue.
// Persistent: CTA i handles tiles i, i + grid, ...
#pragma once
#include "tc_ptx.cuh"
#include <cuda_bf16.h>

struct TcConvParams {
  const float* bias;
  int taps, pad, P;          // kernel taps, left padding, stride
  int kblocks;               // C_in / 64
  int n_tiles;               // C_out / BN
  int t_blks, T_box, B_box;  // tile = T_box rows of B_box windows (T_box * B_box = 128)
  int num_tiles;
  int relu, has_res;
};

template <int BN> struct TcCfg {
  static constexpr int A_BYTES = 128 * 128;
  static constexpr int B_BYTES = BN * 128;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int OUT_BYTES = 128 * 128;                 // one 64-channel chunk of the output tile
  static constexpr int STAGES = (BN == 256) ? 4 : (BN == 128 ? 6 : 8);
  static constexpr int SMEM = STAGES * STAGE_BYTES + 2 * OUT_BYTES + 1024 /*align*/ + 256 /*barriers*/;
};

__device__ __forceinline__ int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

template <int BN>
__global__ void __launch_bounds__(192, 1)
conv_tc_kernel(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_w,
               const __grid_constant__ CUtensorMap tm_out, const __grid_constant__ CUtensorMap tm_res,
               const TcConvParams p) {
  using Cfg = TcCfg<BN>;
  constexpr int STAGES = Cfg::STAGES;
  extern __shared__ unsigned char smem_raw[];
  const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t out_base = base + STAGES * Cfg::STAGE_BYTES;
  const uint32_t bar_base = out_base + 2 * Cfg::OUT_BYTES;
  // barriers (8 B each): full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2], res_full[2]; then tmem ptr
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  auto res_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 4 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 6);
  unsigned char* gen_base = smem_raw + (base - smem_u32(smem_raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_in); tma_prefetch_desc(&tm_w); tma_prefetch_desc(&tm_out);
    if (p.has_res) tma_prefetch_desc(&tm_res);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 128); mbar_init(res_bar(a), 1); }
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(gen_base + (tmem_slot - base));

  const int kiters = p.taps * p.kblocks;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        const int n_idx = tile % p.n_tiles, m_idx = tile / p.n_tiles;
        const int t0 = (m_idx % p.t_blks) * p.T_box, b0 = (m_idx / p.t_blks) * p.B_box, n0 = n_idx * BN;
        for (int d = 0; d < p.taps; ++d) {
          const int sft = d - p.pad;
          const int toff = floor_div(sft, p.P);
          const int par = sft - toff * p.P;
          for (int kb = 0; kb < p.kblocks; ++kb) {
            mbar_wait(empty_bar(stage), phase ^ 1u);
            mbar_arrive_expect_tx(full_bar(stage), Cfg::STAGE_BYTES);
            const uint32_t sa = base + stage * Cfg::STAGE_BYTES;
            tma_load_4d(sa, &tm_in, full_bar(stage), kb * 64, par, t0 + toff, b0);
            tma_load_3d(sa + Cfg::A_BYTES, &tm_w, full_bar(stage), kb * 64, n0, d);
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (one thread) =====
    if (lane == 0) {
      constexpr uint32_t idesc = umma_idesc_bf16(BN);
      int stage = 0; uint32_t phase = 0;
      int acc = 0; uint32_t acc_phase = 0;
      for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
        mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(acc * 256);
        for (int it = 0; it < kiters; ++it) {
          mbar_wait(full_bar(stage), phase);
          tc_fence_after();
          const uint32_t sa = base + stage * Cfg::STAGE_BYTES;
          const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + Cfg::A_BYTES);
#pragma unroll
          for (int k = 0; k < 4; ++k)   // 4 x (K = 16 bf16 = 32 B) inside the 128-byte swizzle row
            umma_bf16(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), idesc, (it > 0 || k > 0) ? 1u : 0u);
          umma_commit(empty_bar(stage));           // frees the smem slot when these MMAs retire
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
        umma_commit(tfull_bar(acc));               // accumulator complete -> epilogue
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
    }
  } else {
    // ===== epilogue: 4 warps, thread <-> one output row =====
    const int q = warp & 3;                        // TMEM lane quadrant this warp may access
    const int row = q * 32 + lane;
    const bool leader = (threadIdx.x == 64);
    int acc = 0; uint32_t acc_phase = 0;
    uint32_t chunk_ctr = 0;
    for (int tile = blockIdx.x; tile < p.num_tiles; tile += gridDim.x) {
      const int n_idx = tile % p.n_tiles, m_idx = tile / p.n_tiles;
      const int t0 = (m_idx % p.t_blks) * p.T_box, b0 = (m_idx / p.t_blks) * p.B_box, n0 = n_idx * BN;
      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
#pragma unroll 1
      for (int c = 0; c < BN / 64; ++c, ++chunk_ctr) {
        const int buf = chunk_ctr & 1u;
        const uint32_t sbuf = out_base + buf * Cfg::OUT_BYTES;
        if (leader) {
          tma_store_wait_read<1>();                // the store that last used this buffer has read it
          if (p.has_res) {
            mbar_arrive_expect_tx(res_bar(buf), Cfg::OUT_BYTES);
            tma_load_4d(sbuf, &tm_res, res_bar(buf), n0 + c * 64, 0, t0, b0);
          }
        }
        named_bar_sync(1, 128);
        uint32_t v[64];
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * 256 + c * 64);
        tmem_ld32(taddr, v);
        tmem_ld32(taddr + 32, v + 32);
        tmem_ld_wait();
        if (c == BN / 64 - 1) {                    // accumulator drained: hand it back to the MMA warp
          tc_fence_before();
          mbar_arrive(tempty_bar(acc));
        }
        if (p.has_res) mbar_wait(res_bar(buf), (chunk_ctr >> 1) & 1u);
        const float4* bias4 = reinterpret_cast<const float4*>(p.bias + n0 + c * 64);
        unsigned char* rowp = gen_base + (sbuf - base) + row * 128;
#pragma unroll
        for (int j = 0; j < 8; ++j) {              // 8 pieces of 8 channels (16 B of bf16)
          const float4 bA = __ldg(bias4 + 2 * j), bB = __ldg(bias4 + 2 * j + 1);
          float f[8];
          f[0] = __uint_as_float(v[8 * j + 0]) + bA.x; f[1] = __uint_as_float(v[8 * j + 1]) + bA.y;
          f[2] = __uint_as_float(v[8 * j + 2]) + bA.z; f[3] = __uint_as_float(v[8 * j + 3]) + bA.w;
          f[4] = __uint_as_float(v[8 * j + 4]) + bB.x; f[5] = __uint_as_float(v[8 * j + 5]) + bB.y;
          f[6] = __uint_as_float(v[8 * j + 6]) + bB.z; f[7] = __uint_as_float(v[8 * j + 7]) + bB.w;
          uint4* sp = reinterpret_cast<uint4*>(rowp + ((j ^ (row & 7)) << 4));   // 128B-swizzle position
          if (p.has_res) {
            const uint4 r = *sp;
            const __nv_bfloat162* rb = reinterpret_cast<const __nv_bfloat162*>(&r);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const float2 rf = __bfloat1622float2(rb[e]);
              f[2 * e] += rf.x; f[2 * e + 1] += rf.y;
            }
          }
          if (p.relu) {
#pragma unroll
            for (int e = 0; e < 8; ++e) f[e] = fmaxf(f[e], 0.f);
          }
          uint4 o;
          __nv_bfloat162* ob = reinterpret_cast<__nv_bfloat162*>(&o);
#pragma unroll
          for (int e = 0; e < 4; ++e) ob[e] = __floats2bfloat162_rn(f[2 * e], f[2 * e + 1]);
          *sp = o;
        }
        fence_proxy_async_smem();                  // generic-proxy writes -> visible to the TMA store
        named_bar_sync(1, 128);
        if (leader) {
          tma_store_4d(&tm_out, sbuf, n0 + c * 64, 0, t0, b0);
          tma_store_commit();
        }
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
    }
    if (leader) tma_store_wait_all<0>();
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 512); }
}
