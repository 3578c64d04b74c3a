// Fused basic block of the 64-channel stage (hard part 3): conv3+norm+ReLU -> conv3+norm -> +x -> ReLU
// in ONE kernel, so the intermediate tensor and the residual never leave the SM.
//
//   y1[t] = relu(ba + sum_d Wa[d] x[t + d - 1])          (rows outside [0, T) are ZERO: conv_b's 'same' padding)
//   y2[t] = relu(bb + sum_d Wb[d] y1[t + d - 1] + x[t])
//
// Tile = 126 output rows of one window.  Per tile:
//   X  : one TMA box of 130 input rows (t0 - 2 .. t0 + 127, out-of-range rows zero-filled), SWIZZLE_128B
//   MMA_a (M128 N64 K16 x 12): tap d reads X through a descriptor shifted by d rows  -> acc_a row r = y1[t0 - 1 + r]
//   epilogue A : acc_a + ba -> fp16 -> ReLU -> zero the rows outside the window -> Y tile in shared memory (same
//                swizzled layout, i.e. directly an A operand)
//   MMA_b : tap d reads Y shifted by d rows                                          -> acc_b row r = y2[t0 + r], r < 126
//   epilogue B : acc_b + bb + x (X rows r + 2, still in shared memory) -> fp16 -> ReLU -> staging -> TMA store (126 rows)
// HBM traffic per block: x read once, y2 written once (the unfused pair reads 3 tensors and writes 2).
// Both weight sets (2 x 24 KB) stay resident.  Rings: X (NX slots), Y (NY), staging (NO); TMEM: 2 + 2 accumulators.
//
// Warp roles (18 warps): 0 TMA producer, 1 MMA issuer (+TMEM), 2-9 two epilogue-A groups, 10-17 two epilogue-B groups;
// group g of either kind takes this CTA's tiles g, g + 2, ... (= accumulator stage g): one 128 x 64 epilogue costs about
// three times the tile's MMA time, so each kind needs two groups in flight to keep up.
#pragma once
#include "conv_tc_kernel.cuh"

struct TcBlockParams {
  const float* bias_a;
  const float* bias_b;
  int T;                 // rows per window
  int tiles_per_win;     // ceil(T / 126)
  int num_tiles;         // windows * tiles_per_win
  TcFastDiv div_tw;      // by tiles_per_win
  int nx, ny, no;        // ring depths
  int reverse;           // walk the tiles from the last to the first
  // shared stem (stem_bf16.cu): tm_x is a strided view of the stem of the whole stream; rows 0, 1 and T - 1 of every window
  // are overwritten in shared memory with the window's own edge rows [windows][3][64] before the tile is used (null = off)
  const af_act_t* edge;
  // shared stage (conv_tc.cu): a batch of short windows stored back to back, zero_valid data rows + separator rows per
  // zero_period rows: y1 is forced to zero on the separators so that they act as each short window's zero padding
  int zero_period, zero_valid;   // 0 = off
#ifdef AFRAME_TC_CYCLES
  long long* dbg_out;    // experiments build only: per-role cycle counters of CTA 0 (null = off)
#endif
};

#define TCB_ROWS 126
#define TCB_SLOT (17 * 1024)          // 130 rows x 128 B, padded to the swizzle period
#define TCB_W_BYTES (3 * 64 * 128)    // one conv's resident weights
#define TCB_FIXED 3072
__host__ __device__ constexpr int tcb_smem(int nx, int ny, int no) {
  return TCB_FIXED + 2 * TCB_W_BYTES + (nx + ny) * TCB_SLOT + 2 * no * TC_OUT_BYTES;   // no staging slots per B group
}

__global__ void __launch_bounds__(576, 1)
conv_block_kernel(const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_wa,
                  const __grid_constant__ CUtensorMap tm_wb, const __grid_constant__ CUtensorMap tm_out,
                  const TcBlockParams p) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const uint32_t base = smem_u32(smem_raw);
  if (base & 1023u) __trap();
  const int NX = p.nx, NY = p.ny, NO = p.no;
  // barriers: x_full[NX] x_empty[NX] y_full[NY] y_empty[NY] a_full[2] a_empty[2] b_full[2] b_empty[2] w_bar, tmem slot
  auto x_full = [&](int s) { return base + 8u * s; };
  auto x_empty = [&](int s) { return base + 8u * (NX + s); };
  auto y_full = [&](int s) { return base + 8u * (2 * NX + s); };
  auto y_empty = [&](int s) { return base + 8u * (2 * NX + NY + s); };
  const uint32_t bar2 = base + 8u * (2 * NX + 2 * NY);
  auto a_full = [&](int s) { return bar2 + 8u * s; };
  auto a_empty = [&](int s) { return bar2 + 8u * (2 + s); };
  auto b_full = [&](int s) { return bar2 + 8u * (4 + s); };
  auto b_empty = [&](int s) { return bar2 + 8u * (6 + s); };
  const uint32_t w_bar = bar2 + 8u * 8;
  const uint32_t tmem_slot = w_bar + 8u;
  auto x_tma = [&](int s) { return tmem_slot + 8u + 8u * s; };   // edge mode: TMA completion, before the patch
  float* s_ba = reinterpret_cast<float*>(smem_raw + 512);
  float* s_bb = s_ba + 64;
  const uint32_t wa_base = base + TCB_FIXED, wb_base = wa_base + TCB_W_BYTES;
  const uint32_t xs_base = wb_base + TCB_W_BYTES;
  const uint32_t ys_base = xs_base + NX * TCB_SLOT;
  const uint32_t os_base = ys_base + NY * TCB_SLOT;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_x); tma_prefetch_desc(&tm_wa); tma_prefetch_desc(&tm_wb); tma_prefetch_desc(&tm_out);
    for (int s = 0; s < NX; ++s) { mbar_init(x_full(s), 1); mbar_init(x_empty(s), 2); mbar_init(x_tma(s), 1); }   // x_empty: MMA_a commit + epilogue B
    for (int s = 0; s < NY; ++s) { mbar_init(y_full(s), 4); mbar_init(y_empty(s), 1); }   // 4 epilogue-A warps | MMA_b commit
    for (int s = 0; s < 2; ++s) {
      mbar_init(a_full(s), 1); mbar_init(a_empty(s), 4);
      mbar_init(b_full(s), 1); mbar_init(b_empty(s), 4);
    }
    mbar_init(w_bar, 1);
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc(tmem_slot, 256);
  if (threadIdx.x < 64) { s_ba[threadIdx.x] = p.bias_a[threadIdx.x]; s_bb[threadIdx.x] = p.bias_b[threadIdx.x]; }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - base));
  pdl_launch_dependents();

  auto decode = [&](int tile, int& b, int& t0) {
    int i;
    if (p.reverse) tile = p.num_tiles - 1 - tile;
    p.div_tw.divmod(tile, b, i);
    t0 = i * TCB_ROWS;
  };
  const int first = blockIdx.x, step = gridDim.x;
#ifdef AFRAME_TC_CYCLES
  const bool prof = p.dbg_out != nullptr && blockIdx.x == 0;
  long long tprev = prof ? clock64() : 0, tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  auto T = [&](int slot) { if (prof) { const long long t = clock64(); tacc[slot] += t - tprev; tprev = t; } };
  auto Tflush = [&](int role) { if (prof) for (int i = 0; i < 8; ++i) p.dbg_out[role * 8 + i] = tacc[i]; };
#else
  auto T = [](int) {};
  auto Tflush = [](int) {};
#endif

  if (warp == 0) {
    // ===== TMA producer =====
    if (elect_one()) {
      mbar_arrive_expect_tx(w_bar, 2 * TCB_W_BYTES);
      for (int d = 0; d < 3; ++d) {
        tma_load_3d(wa_base + d * 8192, &tm_wa, w_bar, 0, 0, d);
        tma_load_3d(wb_base + d * 8192, &tm_wb, w_bar, 0, 0, d);
      }
    }
    __syncwarp();
    pdl_wait();                                    // x is the previous layer's output
    if (p.edge == nullptr) {
    int slot = 0; uint32_t ph = 0;
    for (int tile = first; tile < p.num_tiles; tile += step) {
      int b, t0;
      decode(tile, b, t0);
      T(0);
      mbar_wait(x_empty(slot), ph ^ 1u);
      T(1);
      if (elect_one()) {
        mbar_arrive_expect_tx(x_full(slot), 130 * 128);
        tma_load_3d(xs_base + slot * TCB_SLOT, &tm_x, x_full(slot), 0, t0 - 2, b);
      }
      __syncwarp();
      if (++slot == NX) { slot = 0; ph ^= 1u; }
      T(2);
    }
    } else {
      // edge mode: issue whatever slot is free, and hand a tile to the MMA warp (x_full) once its TMA has landed and the
      // window's own rows 0, 1, T - 1 -- where the box holds them -- have been written over the stream's values
      int n_my = 0;
      for (int tile = first; tile < p.num_tiles; tile += step) ++n_my;
      int slot = 0, fslot = 0, n_issued = 0, n_final = 0;
      uint32_t ph = 0, fph = 0;
      while (n_final < n_my) {
        bool did = false;
        if (n_issued < n_my && __all_sync(0xffffffffu, mbar_test(x_empty(slot), ph ^ 1u))) {
          int b, t0;
          decode(first + n_issued * step, b, t0);
          if (elect_one()) {
            mbar_arrive_expect_tx(x_tma(slot), 130 * 128);
            tma_load_3d(xs_base + slot * TCB_SLOT, &tm_x, x_tma(slot), 0, t0 - 2, b);
          }
          __syncwarp();
          if (++slot == NX) { slot = 0; ph ^= 1u; }
          ++n_issued; did = true;
        }
        if (n_final < n_issued && __all_sync(0xffffffffu, mbar_test(x_tma(fslot), fph))) {
          int b, t0;
          decode(first + n_final * step, b, t0);
          const int k = lane >> 3, jj = lane & 7;          // lanes 8k .. 8k+7: edge row k, 16-byte piece jj
          const int t = k < 2 ? k : p.T - 1;
          const int xr = t - t0 + 2;                       // row of the box that holds window row t
          if (k < 3 && xr >= 0 && xr < 130 && !(k == 1 && p.T < 2)) {
            const uint4 v = *reinterpret_cast<const uint4*>(p.edge + ((int64_t)b * 3 + k) * 64 + jj * 8);
            *reinterpret_cast<uint4*>(smem_raw + (xs_base - base) + fslot * TCB_SLOT + xr * 128 + ((jj ^ (xr & 7)) << 4)) = v;
          }
          fence_proxy_async_smem();                        // generic-proxy writes -> visible to the tensor core's reads
          __syncwarp();
          if (elect_one()) mbar_arrive(x_full(fslot));
          __syncwarp();
          if (++fslot == NX) { fslot = 0; fph ^= 1u; }
          ++n_final; did = true;
        }
        if (!did) __nanosleep(20);
      }
    }
    if (lane == 0) Tflush(0);
  } else if (warp == 1) {
    // ===== MMA issuer (whole warp runs the uniform loop, one elected lane issues) =====
    constexpr uint32_t idesc = umma_idesc_f16_mn(128, 64);
    mbar_wait(w_bar, 0);
    int n_my = 0;
    for (int tile = first; tile < p.num_tiles; tile += step) ++n_my;
    // Issue whatever is ready: A(i) needs its X tile and a free accumulator, B(j) needs the y1 tile written by
    // epilogue A(j).  A fixed A(i), B(i-1) order would stall every iteration for one full epilogue-A latency.
    const uint32_t xs_lo = umma_desc_lo(xs_base), ys_lo = umma_desc_lo(ys_base);
    const uint32_t wa_lo = umma_desc_lo(wa_base), wb_lo = umma_desc_lo(wb_base);
    int ia = 0, jb = 0;
    while (jb < n_my) {
      bool did = false;
      T(0);
      if (ia < n_my) {
        const int xs = ia % NX, as = ia & 1;
        const bool ok = mbar_test(x_full(xs), (uint32_t)((ia / NX) & 1)) && mbar_test(a_empty(as), (uint32_t)(((ia >> 1) & 1) ^ 1));
        if (__all_sync(0xffffffffu, ok)) {
          tc_fence_after();
          if (elect_one()) {
            const uint32_t d_tmem = tmem_base + (uint32_t)(as * 64);
            const uint32_t a_lo = xs_lo + (uint32_t)xs * (TCB_SLOT >> 4);
            umma_mma_lohi<false>(d_tmem, a_lo, wa_lo, idesc);
#pragma unroll
            for (int m = 1; m < 12; ++m)           // tap d = m / 4 (8 = one 128-byte row), K step k = m % 4 (2 = 32 bytes)
              umma_mma_lohi<true>(d_tmem, a_lo + (m / 4) * 8 + (m % 4) * 2, wa_lo + (m / 4) * 512 + (m % 4) * 2, idesc);
            umma_commit(a_full(as));
            umma_commit(x_empty(xs));              // first of the slot's two releases
          }
          __syncwarp();
          ++ia; did = true;
          T(1);
        }
      }
      if (jb < ia) {
        const int ys = jb % NY, bs = jb & 1;
        const bool ok = mbar_test(y_full(ys), (uint32_t)((jb / NY) & 1)) && mbar_test(b_empty(bs), (uint32_t)(((jb >> 1) & 1) ^ 1));
        if (__all_sync(0xffffffffu, ok)) {
          tc_fence_after();
          if (elect_one()) {
            const uint32_t d_tmem = tmem_base + (uint32_t)(128 + bs * 64);
            const uint32_t a_lo = ys_lo + (uint32_t)ys * (TCB_SLOT >> 4);
            umma_mma_lohi<false>(d_tmem, a_lo, wb_lo, idesc);
#pragma unroll
            for (int m = 1; m < 12; ++m)
              umma_mma_lohi<true>(d_tmem, a_lo + (m / 4) * 8 + (m % 4) * 2, wb_lo + (m / 4) * 512 + (m % 4) * 2, idesc);
            umma_commit(b_full(bs));
            umma_commit(y_empty(ys));
          }
          __syncwarp();
          ++jb; did = true;
          T(2);
        }
      }
      if (!did) { __nanosleep(20); T(3); }
    }
    if (lane == 0) Tflush(1);
  } else {
    const int q = warp & 3;                        // TMEM lane quadrant of this warp
    const int row = q * 32 + lane;
    const bool grp_b = warp >= 10;
    const int g = ((warp - 2) >> 2) & 1;           // group of its kind: tiles g, g + 2, ...
    const __half2 z2 = __float2half2_rn(0.f);
    auto pack_relu = [&](float a, float b) -> uint32_t {   // fp16 (RNE, saturating), then ReLU
      const uint32_t pk = af_act_pack2(a, b);
      const __half2 m = __hmax2(*reinterpret_cast<const __half2*>(&pk), z2);
      return *reinterpret_cast<const uint32_t*>(&m);
    };
    if (!grp_b) {
      // ===== epilogue A: acc_a -> y1 tile (an A operand of conv_b) =====
      const float4* bias4 = reinterpret_cast<const float4*>(s_ba);
      int i = g;
      for (int tile = first + g * step; tile < p.num_tiles; tile += 2 * step, i += 2) {
        int b, t0;
        decode(tile, b, t0);
        const int as = i & 1, ys = i % NY;
        T(0);
        mbar_wait(a_full(as), (uint32_t)((i >> 1) & 1));
        T(1);
        tc_fence_after();
        uint32_t v[64];
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(as * 64);
        tmem_ld32(taddr, v);
        tmem_ld32(taddr + 32, v + 32);
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(a_empty(as));
        const int t = t0 - 1 + row;                // y1 row held by this thread
        bool inside = t >= 0 && t < p.T;
        if (p.zero_period > 0 && inside) inside = (t % p.zero_period) < p.zero_valid;
        T(2);
        mbar_wait(y_empty(ys), (uint32_t)(((i / NY) & 1) ^ 1));   // MMA_b of the tile that last used the slot is done
        T(3);
        unsigned char* rowp = smem_raw + (ys_base - base) + ys * TCB_SLOT + row * 128;
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {
          const float4 bA = bias4[2 * jj], bB = bias4[2 * jj + 1];
          uint4 o;
          o.x = pack_relu(__uint_as_float(v[8 * jj + 0]) + bA.x, __uint_as_float(v[8 * jj + 1]) + bA.y);
          o.y = pack_relu(__uint_as_float(v[8 * jj + 2]) + bA.z, __uint_as_float(v[8 * jj + 3]) + bA.w);
          o.z = pack_relu(__uint_as_float(v[8 * jj + 4]) + bB.x, __uint_as_float(v[8 * jj + 5]) + bB.y);
          o.w = pack_relu(__uint_as_float(v[8 * jj + 6]) + bB.z, __uint_as_float(v[8 * jj + 7]) + bB.w);
          if (!inside) o = make_uint4(0u, 0u, 0u, 0u);
          *reinterpret_cast<uint4*>(rowp + ((jj ^ (row & 7)) << 4)) = o;
        }
        T(4);
        fence_proxy_async_smem();                  // generic-proxy writes -> visible to the tensor core's smem reads
        __syncwarp();
        if (lane == 0) mbar_arrive(y_full(ys));
        T(5);
      }
      if (((warp - 2) & 3) == 0 && lane == 0) Tflush(2 + g);
    } else {
      // ===== epilogue B: acc_b + bias + x -> fp16 -> ReLU -> staging -> TMA store of 126 rows =====
      const float4* bias4 = reinterpret_cast<const float4*>(s_bb);
      const bool leader = ((warp - 2) & 3) == 0 && lane == 0;
      const uint32_t og_base = os_base + (uint32_t)(g * NO) * TC_OUT_BYTES;   // this group's staging slots
      int i = g;
      for (int tile = first + g * step; tile < p.num_tiles; tile += 2 * step, i += 2) {
        int b, t0;
        decode(tile, b, t0);
        const int bs = i & 1, xs = i % NX, os = (i >> 1) % NO;
        T(0);
        mbar_wait(b_full(bs), (uint32_t)((i >> 1) & 1));
        T(1);
        tc_fence_after();
        uint32_t v[64];
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(128 + bs * 64);
        tmem_ld32(taddr, v);
        tmem_ld32(taddr + 32, v + 32);
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(b_empty(bs));
        T(2);
        if (leader) tma_store_wait_read_n(NO - 1);                 // staging slot of this tile is free again
        named_bar_sync(1 + g, 128);
        T(3);
        // residual x[t0 + row] = X row (row + 2); rows 126, 127 of the tile are not part of the output
        const int xr = row + 2 < 130 ? row + 2 : 129;
        const unsigned char* xrow = smem_raw + (xs_base - base) + xs * TCB_SLOT + xr * 128;
        unsigned char* orow = smem_raw + (og_base - base) + os * TC_OUT_BYTES + row * 128;
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {
          const float4 bA = bias4[2 * jj], bB = bias4[2 * jj + 1];
          const uint4 r = *reinterpret_cast<const uint4*>(xrow + ((jj ^ (xr & 7)) << 4));
          const uint32_t rw[4] = {r.x, r.y, r.z, r.w};
          float f[8];
          f[0] = __uint_as_float(v[8 * jj + 0]) + bA.x; f[1] = __uint_as_float(v[8 * jj + 1]) + bA.y;
          f[2] = __uint_as_float(v[8 * jj + 2]) + bA.z; f[3] = __uint_as_float(v[8 * jj + 3]) + bA.w;
          f[4] = __uint_as_float(v[8 * jj + 4]) + bB.x; f[5] = __uint_as_float(v[8 * jj + 5]) + bB.y;
          f[6] = __uint_as_float(v[8 * jj + 6]) + bB.z; f[7] = __uint_as_float(v[8 * jj + 7]) + bB.w;
          uint4 o;
          uint32_t* ow = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float2 xr2 = af_act_unpack2(rw[e]);
            ow[e] = pack_relu(f[2 * e] + xr2.x, f[2 * e + 1] + xr2.y);
          }
          *reinterpret_cast<uint4*>(orow + ((jj ^ (row & 7)) << 4)) = o;
        }
        T(4);
        fence_proxy_async_smem();
        named_bar_sync(1 + g, 128);                // all 128 rows staged, all residual reads of the X slot done
        if (leader) {
          mbar_arrive(x_empty(xs));                // second of the slot's two releases
          tma_store_3d(&tm_out, og_base + os * TC_OUT_BYTES, 0, t0, b);
          tma_store_commit();
        }
        T(5);
      }
      if (leader) Tflush(4 + g);
      if (leader) tma_store_wait_all<0>();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) { tc_fence_after(); tmem_dealloc(tmem_base, 256); }
}
