// 1D convolution (k = 1 or 3, stride 1 or 2) as an implicit GEMM on the 5th-gen tensor cores.
//
//   out[b][t][co] = relu( bias[co] + sum_{d, ci} W'[d][co][ci] * in[b][P*t + d - pad][ci] (+ res[b][t][co]) )
//
//   GEMM view: M = (window, t) rows, N = C_out, K = taps * C_in.  Activations are channels-last fp16, so a
//   row of A for tap d is the contiguous channel vector of input row P*t + d - pad.
//   A tile (128 rows x 64 ch) : ONE TMA box of the rank-4 view (C_in, P, T_in/P, B), start row shifted per
//                               tap; out-of-range rows (t = -1, T) are zero-filled by TMA = 'same' padding,
//                               per window, so rows never bleed between windows.  Stride 2 = parity dim.
//   B tile (BN x 64 ch)       : TMA box of the folded fp16 weights [taps][C_out][C_in] (K-major).
//   tcgen05.mma kind::f16 (fp16 activations x fp16 weights) M=128, N=BN, K=16, fp32 accumulators in TMEM
//   (two stages of BN columns).
//   Epilogue: tcgen05.ld -> +bias (+residual, prefetched by TMA) -> fp16 -> ReLU -> swizzled smem -> TMA store,
//   or (HEAD) the fused global-average-pool + linear head: per-(window, slab) partial dot products.
//
// Warp roles: warp 0 TMA producer, warp 1 MMA issuer (+TMEM alloc), then EG epilogue groups of 4 warps (CTA pairs: 8 warps,
// two per TMEM lane quadrant, each taking half of a chunk's columns), then one store warp per epilogue group (storing
// variants): it issues the group's TMA stores and residual prefetches, so the epilogue threads never wait on a store.
// With EG = 2 the groups take alternate tiles (group g <-> TMEM accumulator stage g), which doubles the
// epilogue rate of the small-K layers whose epilogue, not the MMA, is the critical path.
// Persistent: CTA i handles tiles i, i + grid, ...
#pragma once
#include "tc_ptx.cuh"
#include "common.cuh"

// Division by a run-time constant without the ~200-cycle integer-divide sequence (the tile loops of the producer,
// MMA and epilogue roles are single dependent instruction streams): q = (umulhi(x, mul) + x) >> shr, exact for
// 0 <= x < 2^31 (Granlund-Montgomery round-up method; mul, shr computed on the host by tc_fastdiv).
struct TcFastDiv {
  uint32_t mul, shr, d;
  __device__ __forceinline__ void divmod(int x, int& q, int& r) const {
    q = (int)(((uint64_t)__umulhi((uint32_t)x, mul) + (uint32_t)x) >> shr);
    r = x - q * (int)d;
  }
};
static inline TcFastDiv tc_fastdiv(uint32_t d) {
  TcFastDiv f; f.d = d; f.shr = 0;
  while ((1ull << f.shr) < d) ++f.shr;
  f.mul = (uint32_t)((((1ull << f.shr) - d) << 32) / d + 1);
  return f;
}

struct TcConvParams {
  const float* bias;
  TcFastDiv div_n, div_t;    // by n_tiles and by t_blks
  TcFastDiv div_tbox;        // by T_box
  int tap_toff[3], tap_par[3];   // per tap: row offset and parity plane of the strided input view
  int taps, pad, P;          // kernel taps, left padding, stride
  int kblocks;               // C_in / 64
  int n_tiles;               // C_out / BN
  int t_blks, T_box, B_box;  // tile = T_box rows of B_box windows (T_box * B_box = 128)
  int num_tiles;
  int reverse;               // walk the tiles from the last to the first (see af_forward_bf16: L2 reuse between layers)
  int relu, has_res;
  int stages;                // smem ring depth of the main loop
  int nbuf, pf;              // output/residual staging buffers per epilogue group, residual prefetch distance
  int c_out;
  // fused head (HEAD variant): partial[b][slab][chunk] = sum_{t in slab, c in chunk} fp16(out[b][t][c]) * head_w[c]
  const float* head_w;
  float* head_part;
  int head_slabs;            // T_out / T_box
  // head_rows != 0 (shared stages): head_part receives the dot product of EVERY output row with each head unit instead
  // (unit-major, so that a warp's 32 rows are 32 consecutive floats on both sides):
  // head_part[unit * head_rows_total + (b0 + row / T_box) * head_row_stride + t]; sh_head_rows_kernel sums them per window slab
  int head_rows, head_row_stride;
  long long head_rows_total;
  int64_t nb;                // windows in this launch (head variant bounds check)
  // HALO variant (k = 3, stride 1, whole 128-row tiles inside one window): the folded weights of the layer stay resident
  // in shared memory (w_bytes) and ONE (128 + 2)-row input box per 64-channel block serves all three taps: tap d reads
  // the tile through a shared-memory descriptor whose start address is shifted by d rows (d * 128 B).  Measured on B200:
  // the 128-byte swizzle is applied to the absolute shared-memory address, so the shifted start needs no other change
  // (setting the descriptor's base-offset field to the shift gives wrong results).
  // fused projection shortcut: out += W_sc x_sc, sc_kblocks extra K blocks after the taps, read through tm_res (the
  // strided 1x1 view of the block input) and tm_scw; then has_res = 0 and bias holds b + b_sc.  HALO keeps the shortcut
  // weights resident after the main ones.
  int sc_kblocks;
  // true GroupNorm (NEXT-2): the epilogue also emits, per (window, 32-row slab, unit of gn_unit consecutive channels),
  // the sum and sum of squares of the fp32 accumulators: gn_part[(b * T/32 + slab) * (c_out / gn_unit) + unit]
  float2* gn_part;           // null = off
  int gn_unit;               // min(C / G, 64): 8, 16, 32 or 64
  // shared stages (conv_tc.cu): the launch covers a batch of short windows stored back to back; output rows t with
  // t % zero_period >= zero_valid are separators and are stored as zero (they are the short windows' zero padding)
  int zero_period, zero_valid;   // 0 = off
  int zero_origin;               // the batch of short windows starts at this row (rows before it, a stream, are not masked,
                                 // except the two rows just before it, which are the first short window's padding)
  // packed edge batch (conv_tc.cu, shared stages on the CTA-pair path): the launch covers 2 edge_nbp short windows of edge_P
  // rows each -- windows [0, edge_nbp) hold the first edge_P rows of their window (box at row 0), windows [edge_nbp, 2 edge_nbp)
  // the last edge_P rows (box at row edge_t0_tail = edge_P - T_box) -- and one T_box-row box per short window is computed;
  // the tensor map's zero fill is each window's own padding.  Only the rows within reach of that padding (row < edge_head or
  // row >= edge_T - edge_tail of the window, for THIS layer's output) differ from the stream's; the two rows next to them,
  // which the next layers read as well (a conv reaches one row further, and so does the residual two layers on), are the
  // stream's values edge_stream[(b * edge_shift + row) * c_out ...] (this layer's output over the chunk's stream, written by the
  // previous launch): rows of the box are replaced in the epilogue, rows of the slot outside the box (the box is only as long
  // as the edge rows: T_box = max(edge_head, edge_tail)) are copied global -> global by lanes 1..31 of the store warps (edge_out, cpy_*).
  // The rest of the box is never read.
  int edge_nbp;              // 0 = off; else slots per half (windows + spare slots for the last box of a half)
  int edge_blks_half;        // boxes per half: M tiles [0, edge_blks_half) are window starts, the rest window ends
  int edge_t0_tail, edge_T, edge_P, edge_head, edge_tail;
  int edge_t0_tail_in, edge_t0_tail_sc;   // start of a tail box in the slots it reads (main input / fused-projection input)
  int a_bytes;               // bytes of one activation box (T_box * B_box rows of 128 B; 16 KB unless T_box does not divide 128:
                             // the rest of the 128-row MMA tile is then stale shared memory, and those rows are dropped)
  long long edge_shift;
  const uint4* edge_stream;  // null: nothing is replaced or copied (the stage's last layer: only its edge rows are read)
  uint4* edge_out;           // this launch's slots [2 edge_nbp][edge_P][c_out] (the tensor behind tm_out), for those copies
  int cpy_t0_head, cpy_n_head;   // window rows [cpy_t0, cpy_t0 + cpy_n) of a head / tail slot come from the stream and lie outside
  int cpy_t0_tail, cpy_n_tail;   // the box (cpy_n = 0..2)
  int w_bytes;               // resident weight region (0 unless HALO)
  int stage_bytes;           // bytes per main-loop stage
#ifdef AFRAME_TC_CYCLES      // experiments build only (not compiled into the product library)
  long long* dbg_out;        // per-role cycle counters of CTA 0 (null = off)
#endif
};

// shared-memory carve-up (bytes from the 1024-aligned start of dynamic shared memory):
//   [0, 512) mbarriers + TMEM base slot | [512, 2560) bias[c_out <= 512] | HEAD only: [3072, 5120) head_w
//   then the main-loop ring (1024-aligned stages) and the epilogue staging buffers
#define TC_BAR_BYTES 512
#define TC_OUT_BYTES (128 * 128)    // one 64-channel chunk of the output tile
__host__ __device__ constexpr int tc_fixed_bytes(bool head) { return head ? 5120 : 3072; }

template <int BN, bool CG2 = false> struct TcCfg {
  static constexpr int A_BYTES = 128 * 128;
  static constexpr int B_ROWS = CG2 ? BN / 2 : BN;   // CTA pair: each CTA stages half of the B tile
  static constexpr int B_BYTES = B_ROWS * 128;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
  static constexpr int EG = 2;                       // epilogue groups of 4 warps
  static constexpr bool SPLIT = (BN == 256);         // true: both groups drain every tile (alternate 64-column chunks);
                                                     // false: the groups take alternate tiles
  static constexpr int NACC = 512 / BN;              // TMEM accumulator stages (512 columns)
  // Warps per TMEM lane quadrant in an epilogue group.  CTA pairs (N = 256): two, each taking 32 of a chunk's 64 columns.
  // Their epilogue was the critical path of the 256-channel stage (12 K blocks = 3.1 us of MMA per tile against four
  // 64-column chunks drained by 8 warps that spent their time in latency, not issue: profiles/r02_conv_stage3.md); 16
  // warps halve the time a chunk spends in the epilogue, and 32 accumulator columns per thread fit 576 threads' registers.
  static constexpr int EPW = CG2 ? 2 : 1;
  static constexpr int EPI_COLS = 64 / EPW;          // accumulator columns per epilogue thread and chunk
  static constexpr int GROUP_THREADS = 128 * EPW;
  // One more warp per epilogue group whose only job is that group's TMA traffic (stores of staged chunks, residual
  // prefetch).  With the group's leader thread doing it, 255 threads waited at a named barrier per chunk while one thread
  // waited for the previous store to be read (~900 cycles), decoded the next tile and issued the residual load, and again
  // while it issued the store (~500): profiles/r02_conv_cycles.md.  The store warp and the epilogue threads meet only at
  // mbarriers ("staged": 256 arrivals after the chunk is written; "ready": the buffer is free again / its residual landed).
  static constexpr int STORE_WARPS = EG;
  static constexpr int THREADS = 64 + GROUP_THREADS * EG + 32 * STORE_WARPS;
  static constexpr int smem(int stages, int nbuf, bool head) {
    return tc_fixed_bytes(head) + stages * STAGE_BYTES + EG * nbuf * TC_OUT_BYTES;
  }
  static constexpr int HALO_A_BYTES = 17 * 1024;     // 130 rows x 128 B, padded to the 1024-byte swizzle period
  static constexpr int smem_halo(int stages, int nbuf, int taps, int kblocks) {
    return tc_fixed_bytes(false) + taps * kblocks * BN * 128 + stages * HALO_A_BYTES + EG * nbuf * TC_OUT_BYTES;
  }
};

__device__ __forceinline__ int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// NP x 8 channels (pieces jj0 .. jj0 + NP - 1 of a 64-channel chunk) of one output row: + bias (+ residual read from the
// staging buffer) -> fp16 (RNE, saturating) -> max(., lo) (lo = 0: ReLU, which commutes with the rounding; lo = -inf: none)
// -> staging buffer, or the fused head's dot product.  v holds the NP * 8 accumulator columns.
template <bool RES, bool HEAD, int NP, bool ZR = true>
__device__ __forceinline__ void tc_epilogue_math(const uint32_t* v, const float4* bias4, const float4* hw4,
                                                 unsigned char* rowp, int row, int jj0, __half2 lo2, float& head_acc,
                                                 bool zero_row = false) {
  float hacc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int j = 0; j < NP; ++j) {                   // pieces of 8 channels (16 B of fp16)
    const int jj = jj0 + j;
    const float4 bA = bias4[2 * jj], bB = bias4[2 * jj + 1];
    float f[8];
    f[0] = __uint_as_float(v[8 * j + 0]) + bA.x; f[1] = __uint_as_float(v[8 * j + 1]) + bA.y;
    f[2] = __uint_as_float(v[8 * j + 2]) + bA.z; f[3] = __uint_as_float(v[8 * j + 3]) + bA.w;
    f[4] = __uint_as_float(v[8 * j + 4]) + bB.x; f[5] = __uint_as_float(v[8 * j + 5]) + bB.y;
    f[6] = __uint_as_float(v[8 * j + 6]) + bB.z; f[7] = __uint_as_float(v[8 * j + 7]) + bB.w;
    uint4* sp = reinterpret_cast<uint4*>(rowp + ((jj ^ (row & 7)) << 4));   // 128B-swizzle position
    if (RES) {
      const uint4 r = *sp;
      const uint32_t rw[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {                // fp16 pair -> two fp32 (exact)
        const float2 t = af_act_unpack2(rw[e]);
        f[2 * e] += t.x;
        f[2 * e + 1] += t.y;
      }
    }
    uint4 o;
    uint32_t* ow = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const uint32_t pk = af_act_pack2(f[2 * e], f[2 * e + 1]);
      const __half2 m = __hmax2(*reinterpret_cast<const __half2*>(&pk), lo2);
      ow[e] = *reinterpret_cast<const uint32_t*>(&m);
    }
    if (ZR && zero_row) o = make_uint4(0u, 0u, 0u, 0u);
    if (HEAD) {
      const float4 hA = hw4[2 * jj], hB = hw4[2 * jj + 1];
      const float2 o0 = af_act_unpack2(o.x), o1 = af_act_unpack2(o.y), o2 = af_act_unpack2(o.z), o3 = af_act_unpack2(o.w);
      hacc[0] = fmaf(o0.x, hA.x, hacc[0]); hacc[1] = fmaf(o0.y, hA.y, hacc[1]);
      hacc[2] = fmaf(o1.x, hA.z, hacc[2]); hacc[3] = fmaf(o1.y, hA.w, hacc[3]);
      hacc[0] = fmaf(o2.x, hB.x, hacc[0]); hacc[1] = fmaf(o2.y, hB.y, hacc[1]);
      hacc[2] = fmaf(o3.x, hB.z, hacc[2]); hacc[3] = fmaf(o3.y, hB.w, hacc[3]);
    } else {
      *sp = o;
    }
  }
  if (HEAD) head_acc += (hacc[0] + hacc[1]) + (hacc[2] + hacc[3]);
}

// Sum and sum of squares of the warp's 32 rows x U consecutive accumulator columns, for each of the NV / U units of the
// thread's NV columns; lane 0 stores them (fixed order everywhere: the statistics are reproducible bit for bit).
template <int U, int NV>
__device__ __forceinline__ void tc_gn_partials(const uint32_t* v, float2* dst, int lane) {
#pragma unroll
  for (int k = 0; k < NV / U; ++k) {
    float s = 0.f, q = 0.f;
#pragma unroll
    for (int j = 0; j < U; ++j) { const float x = __uint_as_float(v[k * U + j]); s += x; q = fmaf(x, x, q); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); q += __shfl_xor_sync(0xffffffffu, q, o); }
    if (lane == 0) dst[k] = make_float2(s, q);
  }
}

template <int BN, bool HEAD, bool CG2, bool HALO>
__global__ void __launch_bounds__(TcCfg<BN, CG2>::THREADS, 1)
conv_tc_kernel(const __grid_constant__ CUtensorMap tm_in /* HALO: box of 130 rows */, const __grid_constant__ CUtensorMap tm_w,
               const __grid_constant__ CUtensorMap tm_out, const __grid_constant__ CUtensorMap tm_res /* or shortcut input */,
               const __grid_constant__ CUtensorMap tm_scw /* shortcut weights */, const TcConvParams p,
               // optional second problem (p1.num_tiles > 0; neither HALO nor HEAD): every CTA runs its tiles of the first problem,
               // then its tiles of the second one, through the same pipelines.  The two must be independent (conv_tc.cu pairs a
               // layer's packed edge batch with the next layer's stream) and share BN, ring depth and staging plan.
               const __grid_constant__ CUtensorMap tm_in1, const __grid_constant__ CUtensorMap tm_w1,
               const __grid_constant__ CUtensorMap tm_out1, const __grid_constant__ CUtensorMap tm_res1,
               const __grid_constant__ CUtensorMap tm_scw1, const TcConvParams p1) {
  using Cfg = TcCfg<BN, CG2>;
  constexpr int EG = Cfg::EG;
  constexpr bool SPLIT = Cfg::SPLIT;
  constexpr int NACC = Cfg::NACC;
  // CTA pair (CG2): cluster of 2 CTAs = one M = 256 tile (rows [0,128) in the leader, [128,256) in its peer).
  const uint32_t rank = CG2 ? cluster_ctarank() : 0u;
  const int n_workers = CG2 ? (int)(gridDim.x >> 1) : (int)gridDim.x;   // tile loops step by this
  const int worker = CG2 ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
  // the second problem's tiles are dealt out where the first problem's round-robin stopped, so that no worker takes the odd
  // tile of both (two problems of 5.04 and 1.74 rounds are 7 rounds, not 6 + 2)
  const int worker1 = p1.num_tiles > 0 ? (worker + n_workers - p.num_tiles % n_workers) % n_workers : worker;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const uint32_t base = smem_u32(smem_raw);
  if (base & 1023u) __trap();                      // SWIZZLE_128B tiles need 1024-byte alignment
  unsigned char* gen_base = smem_raw;
  const int STAGES = p.stages;
  // barriers (8 B each): full[S], empty[S], tfull[NACC], tempty[NACC], res[EG][MAXBUF], w_bar; then the TMEM base slot
  auto full_bar = [&](int s) { return base + 8u * s; };
  auto empty_bar = [&](int s) { return base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return base + 8u * (2 * STAGES + NACC + a); };
  constexpr int MAXBUF = 4;
  auto res_bar = [&](int g, int b) { return base + 8u * (2 * STAGES + 2 * NACC + g * MAXBUF + b); };
  const uint32_t w_bar = base + 8u * (2 * STAGES + 2 * NACC + EG * MAXBUF);
  const uint32_t tmem_slot = w_bar + 8u;
  auto staged_bar = [&](int g, int b) { return tmem_slot + 8u + 8u * (g * MAXBUF + b); };
  constexpr bool STW = !HEAD;                      // epilogue groups served by store warps (see TcCfg::STORE_WARPS)
  float* s_bias = reinterpret_cast<float*>(gen_base + TC_BAR_BYTES);
  float* s_headw = reinterpret_cast<float*>(gen_base + 3072);
  static_assert(!HALO || (!CG2 && !HEAD), "HALO is a single-CTA, storing variant");
  const uint32_t w_base = base + tc_fixed_bytes(HEAD);           // HALO: resident weights [tap][kblock][BN rows][128 B]
  const uint32_t stage_base = w_base + (HALO ? p.w_bytes : 0);
  const int STAGE_BYTES = HALO ? p.stage_bytes : Cfg::STAGE_BYTES;
  const uint32_t out_base = stage_base + STAGES * STAGE_BYTES;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tm_in); tma_prefetch_desc(&tm_w);
    if (!HEAD) tma_prefetch_desc(&tm_out);
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < NACC; ++a) {               // tempty: one arrival per epilogue warp that drains the stage
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), (SPLIT ? 8 : 4) * Cfg::EPW * (CG2 ? 2 : 1));
    }
    mbar_init(w_bar, 1);
    for (int g = 0; g < EG; ++g)
      for (int b = 0; b < MAXBUF; ++b) { mbar_init(res_bar(g, b), 1); mbar_init(staged_bar(g, b), Cfg::GROUP_THREADS); }
    if (p.has_res || p.sc_kblocks) tma_prefetch_desc(&tm_res);
    if (p.sc_kblocks) tma_prefetch_desc(&tm_scw);
    fence_mbar_init();
  }
  if (warp == 1) { if (CG2) tmem_alloc_cg2(tmem_slot, 512); else tmem_alloc(tmem_slot, 512); }
  for (int i = threadIdx.x; i < p.c_out; i += blockDim.x) {
    s_bias[i] = p.bias[i];
    if (HEAD) s_headw[i] = p.head_w[i];
  }
  tc_fence_before();
  __syncthreads();
  if (CG2) cluster_sync_all();                     // the peer's barriers exist before any remote arrive / complete_tx
  tc_fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(gen_base + (tmem_slot - base));

  // Programmatic dependent launch: the next layer's CTAs may start their prologue (barriers, TMEM, bias, resident
  // weights) while this grid is still running; everything that reads the previous layer's output comes after pdl_wait().
  pdl_launch_dependents();
  if (!(HALO && warp == 0)) pdl_wait();            // (the halo producer first issues its weight loads, see below)

  const int kiters = p.taps * p.kblocks + p.sc_kblocks;
  // cycle accounting for experiments (CTA 0 only): T(slot) adds the cycles since the previous T() of this thread
#ifdef AFRAME_TC_CYCLES
  const bool prof = p.dbg_out != nullptr && blockIdx.x == 0;
  long long tprev = prof ? clock64() : 0, tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  auto T = [&](int slot) { if (prof) { const long long t = clock64(); tacc[slot] += t - tprev; tprev = t; } };
  auto Tflush = [&](int role) { if (prof) for (int i = 0; i < 8; ++i) p.dbg_out[role * 8 + i] = tacc[i]; };
#else
  auto T = [](int) {};
  auto Tflush = [](int) {};
#endif
  // tile -> (n0, t0, b0): n fastest, then the T_box-row block inside a window group, then the window group
  auto decode = [&](const TcConvParams& p, int tile, int& n_idx, int& t0, int& b0) {
    int mp, tb, bb;
    if (p.reverse) tile = p.num_tiles - 1 - tile;
    p.div_n.divmod(tile, mp, n_idx);
    const int m_idx = mp * (CG2 ? 2 : 1) + (int)rank;
    p.div_t.divmod(m_idx, bb, tb);
    t0 = tb * p.T_box; b0 = bb * p.B_box;
    if (p.edge_nbp > 0 && bb >= p.edge_blks_half) {                  // packed edge batch: window ends, the box ends at the slot's end
      b0 = p.edge_nbp + (bb - p.edge_blks_half) * p.B_box;
      t0 = p.edge_t0_tail;
    }
  };

  if (warp == 0) {
    // ===== TMA producer =====
    // (the whole warp runs the uniform loops; one elected lane issues, so operands stay in uniform registers)
    if (HALO) {
      // resident weights, once per CTA (n_tiles == 1: BN == C_out)
      if (elect_one()) {
        mbar_arrive_expect_tx(w_bar, (uint32_t)p.w_bytes);
        for (int d = 0; d < p.taps; ++d)
          for (int kb = 0; kb < p.kblocks; ++kb)
            tma_load_3d(w_base + (uint32_t)((d * p.kblocks + kb) * BN * 128), &tm_w, w_bar, kb * 64, 0, d);
        for (int kb = 0; kb < p.sc_kblocks; ++kb)
          tma_load_3d(w_base + (uint32_t)((p.taps * p.kblocks + kb) * BN * 128), &tm_scw, w_bar, kb * 64, 0, 0);
      }
      __syncwarp();
      pdl_wait();                                  // the activations below are the previous layer's output
      int stage = 0; uint32_t phase = 0;
      for (int tile = worker; tile < p.num_tiles; tile += n_workers) {
        int n_idx, t0, b0;
        decode(p, tile, n_idx, t0, b0);
        for (int kb = 0; kb < p.kblocks; ++kb) {   // one stage = the 130-row box of one 64-channel block
          T(0);
          mbar_wait(empty_bar(stage), phase ^ 1u);
          T(1);
          const uint32_t sa = stage_base + stage * STAGE_BYTES;
          if (elect_one()) {
            mbar_arrive_expect_tx(full_bar(stage), 130 * 128);
            // rows t0 - 1 .. t0 + 128 of the window; out-of-range rows are zero-filled
            tma_load_4d(sa, &tm_in, full_bar(stage), kb * 64, 0, t0 - 1, b0);
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
          T(2);
        }
        for (int kb = 0; kb < p.sc_kblocks; ++kb) {   // shortcut: the 128 rows x_sc[t0 ..] of one 64-channel block
          mbar_wait(empty_bar(stage), phase ^ 1u);
          if (elect_one()) {
            mbar_arrive_expect_tx(full_bar(stage), 128 * 128);
            tma_load_4d(stage_base + stage * STAGE_BYTES, &tm_res, full_bar(stage), kb * 64, 0, t0, b0);
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
      if (lane == 0) Tflush(0);
    } else {
      const uint32_t lfull0 = CG2 ? mapa_cluster(full_bar(0), 0) : full_bar(0);   // leader's full barriers
      int stage = 0; uint32_t phase = 0;
      auto produce = [&](const CUtensorMap& tm_in, const CUtensorMap& tm_w, const CUtensorMap& tm_res, const CUtensorMap& tm_scw,
                         const TcConvParams& p, int worker) {
      for (int tile = worker; tile < p.num_tiles; tile += n_workers) {
        int n_idx, t0, b0;
        decode(p, tile, n_idx, t0, b0);
        const int n0 = n_idx * BN;
        // packed edge batch, tail boxes: the slots this launch reads may be shorter than the slots it writes
        const bool tail_box = p.edge_nbp > 0 && b0 >= p.edge_nbp;
        const int t0s = tail_box ? p.edge_t0_tail_sc : t0;
        if (tail_box) t0 = p.edge_t0_tail_in;
        // (64-channel block outer, tap inner: the order in which the HALO variant accumulates, so that a layer gives the same
        //  bits whichever of the two computes a row)
        for (int kb = 0; kb < p.kblocks; ++kb) {
          for (int d = 0; d < p.taps; ++d) {
            const int toff = p.tap_toff[d], par = p.tap_par[d];
            T(0);
            mbar_wait(empty_bar(stage), phase ^ 1u);
            T(1);
            const uint32_t sa = stage_base + stage * STAGE_BYTES;
            if (elect_one()) {
              if (CG2) {
                // both CTAs load their own A rows and their half of B; all bytes are counted on the leader's barrier
                if (rank == 0) mbar_arrive_expect_tx(full_bar(stage), 2 * (p.a_bytes + Cfg::B_BYTES));
                const uint32_t lbar = lfull0 + 8u * stage;
                tma_load_4d_cg2(sa, &tm_in, lbar, kb * 64, par, t0 + toff, b0);
                tma_load_3d_cg2(sa + Cfg::A_BYTES, &tm_w, lbar, kb * 64, n0 + (int)rank * Cfg::B_ROWS, d);
              } else {
                mbar_arrive_expect_tx(full_bar(stage), p.a_bytes + Cfg::B_BYTES);
                tma_load_4d(sa, &tm_in, full_bar(stage), kb * 64, par, t0 + toff, b0);
                tma_load_3d(sa + Cfg::A_BYTES, &tm_w, full_bar(stage), kb * 64, n0, d);
              }
            }
            __syncwarp();
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            T(2);
          }
        }
        for (int kb = 0; kb < p.sc_kblocks; ++kb) {   // fused projection shortcut: A from the strided block input
          mbar_wait(empty_bar(stage), phase ^ 1u);
          const uint32_t sa = stage_base + stage * STAGE_BYTES;
          if (elect_one()) {
            if (CG2) {
              if (rank == 0) mbar_arrive_expect_tx(full_bar(stage), 2 * (p.a_bytes + Cfg::B_BYTES));
              const uint32_t lbar = lfull0 + 8u * stage;
              tma_load_4d_cg2(sa, &tm_res, lbar, kb * 64, 0, t0s, b0);
              tma_load_3d_cg2(sa + Cfg::A_BYTES, &tm_scw, lbar, kb * 64, n0 + (int)rank * Cfg::B_ROWS, 0);
            } else {
              mbar_arrive_expect_tx(full_bar(stage), p.a_bytes + Cfg::B_BYTES);
              tma_load_4d(sa, &tm_res, full_bar(stage), kb * 64, 0, t0s, b0);
              tma_load_3d(sa + Cfg::A_BYTES, &tm_scw, full_bar(stage), kb * 64, n0, 0);
            }
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
        }
      }
      };
      produce(tm_in, tm_w, tm_res, tm_scw, p, worker);
      if (!HEAD && p1.num_tiles > 0) produce(tm_in1, tm_w1, tm_res1, tm_scw1, p1, worker1);
      if (lane == 0) Tflush(0);
    }
  } else if (warp == 1) {
    // ===== MMA issuer: the whole warp runs the (uniform) loop, one elected lane issues =====
    if (rank == 0) {
      constexpr uint32_t idesc = umma_idesc_f16_mn(CG2 ? 256 : 128, BN);
      int stage = 0; uint32_t phase = 0;
      int acc = 0; uint32_t acc_phase = 0;
      if (HALO) mbar_wait(w_bar, 0);
      auto issue = [&](const TcConvParams& p, int worker) {
      const int kiters = p.taps * p.kblocks + p.sc_kblocks;
      for (int tile = worker; tile < p.num_tiles; tile += n_workers) {
        T(0);
        mbar_wait(tempty_bar(acc), acc_phase ^ 1u);
        T(1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(acc * BN);
        if (HALO) {
          for (int kb = 0; kb < p.kblocks; ++kb) {
            T(0);
            mbar_wait(full_bar(stage), phase);
            T(2);
            tc_fence_after();
            if (elect_one()) {
              const uint32_t a_lo = umma_desc_lo(stage_base + stage * STAGE_BYTES);
              const uint32_t b_lo = umma_desc_lo(w_base + (uint32_t)(kb * BN * 128));
              const uint32_t b_tap = (uint32_t)(p.kblocks * BN * 128) >> 4;   // weights [tap][kblock][BN rows][128 B]
              // tap d: rows d .. d + 127 of the 130-row box = descriptor start shifted by d rows of 128 B (8 units)
#pragma unroll
              for (int m = 0; m < 12; ++m) {
                const uint32_t al = a_lo + (m / 4) * 8 + (m % 4) * 2, bl = b_lo + (m / 4) * b_tap + (m % 4) * 2;
                if (m == 0 && kb == 0) umma_mma_lohi<false>(d_tmem, al, bl, idesc);
                else umma_mma_lohi<true>(d_tmem, al, bl, idesc);
              }
              umma_commit(empty_bar(stage));
            }
            __syncwarp();
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
            T(3);
          }
          for (int kb = 0; kb < p.sc_kblocks; ++kb) {   // shortcut K block: plain 128-row tile, its resident weights
            mbar_wait(full_bar(stage), phase);
            tc_fence_after();
            if (elect_one()) {
              const uint32_t a_lo = umma_desc_lo(stage_base + stage * STAGE_BYTES);
              const uint32_t b_lo = umma_desc_lo(w_base + (uint32_t)((p.taps * p.kblocks + kb) * BN * 128));
#pragma unroll
              for (int m = 0; m < 4; ++m) umma_mma_lohi<true>(d_tmem, a_lo + m * 2, b_lo + m * 2, idesc);
              umma_commit(empty_bar(stage));
            }
            __syncwarp();
            if (++stage == STAGES) { stage = 0; phase ^= 1u; }
          }
        }
        for (int it = 0; it < (HALO ? 0 : kiters); ++it) {
          T(0);
          mbar_wait(full_bar(stage), phase);
          T(2);
          tc_fence_after();
          const uint32_t sa = stage_base + stage * STAGE_BYTES;
          const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + Cfg::A_BYTES);
          if (elect_one()) {
#pragma unroll
          for (int k = 0; k < 4; ++k) { // 4 x (K = 16 elements = 32 B) inside the 128-byte swizzle row
            if (CG2) umma_mma_cg2(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), idesc, (it > 0 || k > 0) ? 1u : 0u);
            else umma_mma(d_tmem, da + (uint64_t)(2 * k), db + (uint64_t)(2 * k), idesc, (it > 0 || k > 0) ? 1u : 0u);
          }
          if (CG2) umma_commit_cg2(empty_bar(stage), 3);   // frees the smem slot in BOTH CTAs when these MMAs retire
          else umma_commit(empty_bar(stage));
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1u; }
          T(3);
        }
        if (elect_one()) {
          if (CG2) umma_commit_cg2(tfull_bar(acc), 3);   // accumulator complete -> both CTAs' epilogues
          else umma_commit(tfull_bar(acc));
        }
        __syncwarp();
        if (++acc == NACC) { acc = 0; acc_phase ^= 1u; }
        T(4);
      }
      };
      issue(p, worker);
      if (!HALO && !HEAD && p1.num_tiles > 0) issue(p1, worker1);
      if (lane == 0) Tflush(1);
    }
  } else if (warp >= 2 + 4 * Cfg::EPW * EG) {
    // ===== store warp of epilogue group g: lane 0 walks the group's (tile, chunk) sequence over both problems =====
    // (the fused-head variant stores nothing: its store warps are idle)
    const int g = warp - (2 + 4 * Cfg::EPW * EG);
    if (STW && lane == 0) {
      const int NBUF = p.nbuf > 0 ? p.nbuf : 1;
      const uint32_t gbuf = out_base + (uint32_t)(g * NBUF) * TC_OUT_BYTES;
      constexpr int CH = BN / 64;
      // the group's items, as its epilogue threads walk them: SPLIT (N = 256): every tile of this CTA, chunks g, g + 2;
      // else: this CTA's tiles g, g + EG, ..., every chunk
      const int tile_step = (SPLIT ? 1 : EG) * n_workers, tile_first = worker + (SPLIT ? 0 : g) * n_workers;
      const int tile_first1 = worker1 + (SPLIT ? 0 : g) * n_workers;
      constexpr int C_STEP = SPLIT ? 2 : 1;
      const int c_first = SPLIT ? g : 0;
      struct Cur { int prob, tile, c; };
      auto settle = [&](Cur& k) {                  // first valid item at or after k (prob = 2: past the end)
        while (k.prob < 2) {
          const TcConvParams& P = k.prob ? p1 : p;
          if (k.tile < P.num_tiles) return;
          ++k.prob; k.tile = tile_first1; k.c = c_first;
        }
      };
      auto next = [&](Cur& k) {
        k.c += C_STEP;
        if (k.c >= CH) { k.c = c_first; k.tile += tile_step; }
        settle(k);
      };
      // buffer `buf` may be written for item k: its residual tile is on its way, or (no residual) it is simply free
      auto signal_ready = [&](const Cur& k, int buf) {
        if (k.prob >= 2) return;
        const TcConvParams& P = k.prob ? p1 : p;
        if (P.has_res) {
          int n_idx, t0, b0;
          decode(P, k.tile, n_idx, t0, b0);
          mbar_arrive_expect_tx(res_bar(g, buf), P.a_bytes);
          tma_load_4d(gbuf + buf * TC_OUT_BYTES, k.prob ? &tm_res1 : &tm_res, res_bar(g, buf), n_idx * BN + k.c * 64, 0, t0, b0);
        } else {
          mbar_arrive(res_bar(g, buf));
        }
      };
      Cur S = {0, tile_first, c_first}, A = {0, tile_first, c_first};
      settle(S); settle(A);
      for (int i = 0; i < NBUF; ++i) { signal_ready(A, i); next(A); }
      for (uint32_t j = 0; S.prob < 2; ++j) {
        const int buf = j % NBUF;
        mbar_wait(staged_bar(g, buf), (j / NBUF) & 1u);
        const TcConvParams& P = S.prob ? p1 : p;
        int n_idx, t0, b0;
        decode(P, S.tile, n_idx, t0, b0);
        tma_store_4d(S.prob ? &tm_out1 : &tm_out, gbuf + buf * TC_OUT_BYTES, n_idx * BN + S.c * 64, 0, t0, b0);
        tma_store_commit();
        tma_store_wait_read_n(0);                  // the buffer has been read: item j + NBUF may have it
        signal_ready(A, buf);
        next(A); next(S);
      }
      tma_store_wait_all<0>();
    } else if (STW && !HALO) {
      // ===== lanes 1..31 of the store warps (ring variants that store), on their own path: packed edge batch, the stream rows
      // next to each slot's edge rows that the box does not hold (see TcConvParams::edge_out), global -> global, store warp g
      // taking its 1/EG of the tile's columns.  Nothing in this launch reads these rows, so the path meets no barrier.
      auto copy_rows = [&](const TcConvParams& P, int worker) {
        if (P.edge_out == nullptr) return;
        const int cq = P.c_out >> 3;                // uint4 per row
        constexpr int PER_ROW = BN / 8 / EG;        // uint4 of this warp's columns per slot row (a power of two)
        static_assert((PER_ROW & (PER_ROW - 1)) == 0, "PER_ROW");
        for (int tile = worker; tile < P.num_tiles; tile += n_workers) {
          int n_idx, t0, b0;
          decode(P, tile, n_idx, t0, b0);
          const bool tailb = b0 >= P.edge_nbp;
          const int rows_cp = tailb ? P.cpy_n_tail : P.cpy_n_head;
          if (rows_cp <= 0) continue;
          const int tw0 = tailb ? P.cpy_t0_tail : P.cpy_t0_head, bfirst = tailb ? b0 - P.edge_nbp : b0;
          const int srow0 = tw0 - (tailb ? P.edge_T - P.edge_P : 0);
          const int col = ((n_idx * BN) >> 3) + g * PER_ROW;
          const int total = P.B_box * rows_cp * PER_ROW;
          constexpr int NCP = 6;
          for (int i0 = 0; i0 < total; i0 += 31 * NCP) {
            uint4 cr[NCP];
            uint4* cdst[NCP];
#pragma unroll
            for (int k = 0; k < NCP; ++k) {
              const int idx = i0 + (lane - 1) + 31 * k;
              const int srow = idx / PER_ROW, ch = idx % PER_ROW;
              const int slot = srow / rows_cp, r = srow - slot * rows_cp;
              const int b = bfirst + slot;
              cdst[k] = nullptr;
              if (idx < total && b < P.nb) {
                cdst[k] = P.edge_out + ((long long)(tailb ? P.edge_nbp + b : b) * P.edge_P + srow0 + r) * cq + col + ch;
                cr[k] = __ldg(P.edge_stream + ((long long)b * P.edge_shift + tw0 + r) * cq + col + ch);
              }
            }
#pragma unroll
            for (int k = 0; k < NCP; ++k)
              if (cdst[k] != nullptr) *cdst[k] = cr[k];
          }
        }
      };
      copy_rows(p, worker);
      if (p1.num_tiles > 0) copy_rows(p1, worker1);
    }
  } else {
    // ===== epilogue: EG groups of 4 warps, thread <-> one output row =====
    constexpr int EPW = Cfg::EPW, GT = Cfg::GROUP_THREADS, EC = Cfg::EPI_COLS;
    const int ew = warp - 2;
    const int g = ew / (4 * EPW);                  // epilogue group: takes this CTA's tiles g, g + EG, ...
    const int q = warp & 3;                        // TMEM lane quadrant this warp may access
    const int hf = (ew % (4 * EPW)) >> 2;          // which EC columns of a chunk this warp takes (EPW = 2: two warps per quadrant)
    const int row = q * 32 + lane;
    const bool leader = ((ew % (4 * EPW)) == 0) && lane == 0;
    const int NBUF = p.nbuf > 0 ? p.nbuf : 1;      // (the fused head stages nothing)
    const uint32_t gbuf = out_base + (uint32_t)(g * NBUF) * TC_OUT_BYTES;
    constexpr int CH = BN / 64;
    const int tile_step = (SPLIT ? 1 : EG) * n_workers;     // this group's tiles ...
    constexpr int C_STEP = SPLIT ? 2 : 1;                   // ... and its chunks of each tile
    const int c_first = SPLIT ? g : 0;
    const uint32_t tempty_leader0 = CG2 ? mapa_cluster(tempty_bar(0), 0) : tempty_bar(0);

    uint32_t j = 0;                                // chunk counter of this group
    uint32_t seq = SPLIT ? 0 : g;                  // this CTA's tile sequence number
    uint32_t res_par = 0;                          // bit b: phase parity of this group's residual barrier b
    const int PF = p.pf;
    auto drain = [&](const CUtensorMap& tm_out, const CUtensorMap& tm_res, const TcConvParams& p, bool second) {
    const int tile_first = (second ? worker1 : worker) + (SPLIT ? 0 : g) * n_workers;
    if (second) {
      // the second problem's bias replaces the first one's once both groups are done with it; the leader's earlier stores
      // must have read their staging buffers before a residual tile is prefetched into one
      named_bar_sync(3, GT * EG);
      for (int i = (int)threadIdx.x - 64; i < p.c_out; i += GT * EG) s_bias[i] = p.bias[i];
      named_bar_sync(3, GT * EG);
      if (!STW && leader) tma_store_wait_read_n(0);
    }
    int row_bq, row_tq;                            // this thread's row inside the tile's box
    p.div_tbox.divmod(row, row_bq, row_tq);
    // residual prefetch cursor (leader only): item pf_j of this group's (tile, chunk) sequence; the residual tile lands
    // in the staging buffer the chunk's output will be written to (added in place)
    int pf_tile = tile_first, pf_c = c_first;
    uint32_t pf_j = j;
    auto issue_res = [&]() {
      if (pf_tile < p.num_tiles) {
        int n_idx, t0, b0;
        decode(p, pf_tile, n_idx, t0, b0);
        const int buf = pf_j % NBUF;
        mbar_arrive_expect_tx(res_bar(g, buf), p.a_bytes);
        tma_load_4d(gbuf + buf * TC_OUT_BYTES, &tm_res, res_bar(g, buf), n_idx * BN + pf_c * 64, 0, t0, b0);
      }
      ++pf_j;
      pf_c += C_STEP;
      if (pf_c >= CH) { pf_c = c_first; pf_tile += tile_step; }
    };
    if (!STW && leader && p.has_res)
      for (int i = 0; i < PF; ++i) issue_res();

    // packed edge batch: this thread's row of tile (n0_, t0_, b0_) is taken from the stream if it is one of the two rows next to
    // the window's edge rows (the only interior rows a later layer reads): pointer to its first channel of the tile, else null
    auto copy_base = [&](int n0_, int t0_, int b0_) -> const uint4* {
      if (HEAD || p.edge_nbp == 0 || p.edge_stream == nullptr || row >= p.T_box * p.B_box) return nullptr;
      const int m = b0_ + row_bq;                  // short-window slot
      const bool is_tail = m >= p.edge_nbp;
      const int b = is_tail ? m - p.edge_nbp : m;
      const int t_win = (is_tail ? p.edge_T - p.edge_P : 0) + t0_ + row_tq;
      const int d = is_tail ? p.edge_T - p.edge_tail - 1 - t_win : t_win - p.edge_head;   // >= 0: a row of the box past the edge rows
      if (d < 0 || b >= p.nb) return nullptr;
      return p.edge_stream + (((long long)b * p.edge_shift + t_win) * p.c_out + n0_) / 8;
    };
    // ... and is fetched into L1 one tile ahead, so that the epilogue does not wait for L2 (measured: the un-prefetched copy
    // cost the 256-channel stage 30 % of its time)
    auto copy_prefetch = [&](int tile_) {
      if (HEAD || p.edge_nbp == 0 || p.edge_stream == nullptr || tile_ >= p.num_tiles) return;
      int n_i, t0_, b0_;
      decode(p, tile_, n_i, t0_, b0_);
      const uint4* cb = copy_base(n_i * BN, t0_, b0_);
      if (cb != nullptr)
        for (int c = c_first; c < CH; c += C_STEP) asm volatile("prefetch.global.L1 [%0];" :: "l"(cb + c * 8));
    };
    copy_prefetch(tile_first);

    for (int tile = tile_first; tile < p.num_tiles; tile += tile_step, seq += (SPLIT ? 1 : EG)) {
      const int acc = seq % NACC;
      const uint32_t acc_phase = (seq / NACC) & 1u;
      int n_idx, t0, b0;
      decode(p, tile, n_idx, t0, b0);
      const int n0 = n_idx * BN;
      const uint4* copy_tile = copy_base(n0, t0, b0);
      copy_prefetch(tile + tile_step);
      T(0);
      mbar_wait(tfull_bar(acc), acc_phase);
      T(1);
      tc_fence_after();
      float head_acc = 0.f;
#pragma unroll 1
      for (int c = c_first; c < CH; c += C_STEP, ++j) {
        const int buf = j % NBUF;
        const uint32_t sbuf = gbuf + buf * TC_OUT_BYTES;
        if (!STW) {
        if (leader) {
          if (p.has_res) {
            if (!HEAD) tma_store_wait_read_n(NBUF - PF - 1);   // buffer of chunk j + PF is free again
            issue_res();
          } else if (!HEAD) {
            tma_store_wait_read_n(NBUF - 1);                   // buffer of this chunk is free again
          }
        }
        T(2);
        named_bar_sync(1 + g, GT);
        }
        T(3);
        uint32_t v[EC];
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(acc * BN + c * 64 + hf * EC);
        tmem_ld32(taddr, v);
        if (EC == 64) tmem_ld32(taddr + 32, v + 32);
        tmem_ld_wait();
        T(4);
        if (c + C_STEP >= CH) {                    // this group's part of the accumulator is drained: hand it back to the (leader's) MMA warp
          tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            if (CG2) mbar_arrive_cluster(tempty_leader0 + 8u * acc);
            else mbar_arrive(tempty_bar(acc));
          }
        }
        if (!HEAD && p.gn_part != nullptr) {       // (T_box % 32 == 0: the warp's 32 rows are one slab of one window)
          const int r0 = q * 32;
          const int64_t b = b0 + r0 / p.T_box;
          const int slab = (t0 + r0 % p.T_box) >> 5;
          if (b < p.nb) {                          // (gn_unit <= EC: conv_tc.cu)
            float2* dst = p.gn_part + ((b * p.head_slabs + slab) * (int64_t)(p.c_out / p.gn_unit) + (n0 + c * 64 + hf * EC) / p.gn_unit);
            switch (p.gn_unit) {
              case 8: tc_gn_partials<8, EC>(v, dst, lane); break;
              case 16: tc_gn_partials<16, EC>(v, dst, lane); break;
              case 32: tc_gn_partials<32, EC>(v, dst, lane); break;
              default: tc_gn_partials<EC, EC>(v, dst, lane); break;
            }
          }
        }
        if (STW) {                                 // the store warp: this chunk's buffer is free, its residual (if any) has landed
          mbar_wait(res_bar(g, buf), (j / NBUF) & 1u);
        } else if (p.has_res) {                    // (own parity per buffer: with two problems not every chunk has a residual)
          mbar_wait(res_bar(g, buf), (res_par >> buf) & 1u);
          res_par ^= 1u << buf;
        }
        T(5);
        const float4* bias4 = reinterpret_cast<const float4*>(s_bias + n0 + c * 64);
        const float4* hw4 = reinterpret_cast<const float4*>(s_headw + n0 + c * 64);
        unsigned char* rowp = gen_base + (sbuf - base) + row * 128;
        // straight-line code per variant (no run-time branches inside the unrolled loop, so the 8 pieces interleave)
        const __half2 lo2 = __float2half2_rn(p.relu ? 0.f : -INFINITY);
        const int t_row = t0 + row_tq;
        const bool zero_row = p.zero_period > 0 && t_row >= p.zero_origin - 2 &&
                              ((t_row - p.zero_origin + p.zero_period) % p.zero_period) >= p.zero_valid;
        const uint4* copy_row = copy_tile != nullptr ? copy_tile + c * 8 : nullptr;
        constexpr int NP = EC / 8;
        if (p.zero_period > 0) {                   // (row masks exist only in the fixed-length short-window form)
          if (p.has_res) tc_epilogue_math<true, HEAD, NP, true>(v, bias4, hw4, rowp, row, hf * NP, lo2, head_acc, zero_row);
          else tc_epilogue_math<false, HEAD, NP, true>(v, bias4, hw4, rowp, row, hf * NP, lo2, head_acc, zero_row);
        } else {
          if (p.has_res) tc_epilogue_math<true, HEAD, NP, false>(v, bias4, hw4, rowp, row, hf * NP, lo2, head_acc);
          else tc_epilogue_math<false, HEAD, NP, false>(v, bias4, hw4, rowp, row, hf * NP, lo2, head_acc);
        }
        if (!HEAD && copy_row != nullptr) {        // the staged row is replaced by the stream's (independent loads, then the stores)
          uint4 cr[NP];
#pragma unroll
          for (int j = 0; j < NP; ++j) cr[j] = __ldg(copy_row + hf * NP + j);
#pragma unroll
          for (int j = 0; j < NP; ++j) *reinterpret_cast<uint4*>(rowp + (((hf * NP + j) ^ (row & 7)) << 4)) = cr[j];
        }
        if (HEAD) {
          // the warp's 32 rows are one 32-row slab of one window (T_box % 32 == 0): reduce and emit a partial
          float s = head_acc;
          head_acc = 0.f;
          // head units: EC channels (one per epilogue warp of a quadrant), c_out / EC of them per row
          const int hu = (n_idx * CH + c) * EPW + hf, n_hu = (p.c_out >> 6) * EPW;
          if (p.head_rows) {
            // (rows past the tensor -- the peer CTA's half of a last, partial pair tile -- have no place in a unit's row array)
            const long long hr = (long long)(b0 + row / p.T_box) * p.head_row_stride + t_row;
            if (row < p.T_box * p.B_box && t_row < p.head_row_stride && hr < p.head_rows_total) p.head_part[hu * p.head_rows_total + hr] = s;
          } else {
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
          const int r0 = q * 32;
          const int64_t b = b0 + r0 / p.T_box;
          const int slab = (t0 + r0 % p.T_box) >> 5;
          if (lane == 0 && b < p.nb)
            p.head_part[(b * p.head_slabs + slab) * n_hu + hu] = s;
          }
          named_bar_sync(1 + g, GT);               // residual buffer fully read before it is refilled
        } else {
          T(6);
          fence_proxy_async_smem();                // generic-proxy writes -> visible to the TMA store
          if (STW) {
            mbar_arrive(staged_bar(g, buf));       // the store warp takes it from here
          } else {
          named_bar_sync(1 + g, GT);
          if (leader) {
            tma_store_4d(&tm_out, sbuf, n0 + c * 64, 0, t0, b0);
            tma_store_commit();
          }
          }
          T(7);
        }
      }
    }
    };
    drain(tm_out, tm_res, p, false);
    if (!HALO && !HEAD && p1.num_tiles > 0) drain(tm_out1, tm_res1, p1, true);
    if (leader) Tflush(2 + g);
    if (!STW && leader && !HEAD) tma_store_wait_all<0>();
  }
  tc_fence_before();
  __syncthreads();
  if (CG2) cluster_sync_all();                     // the peer has drained its half of the accumulators
  if (warp == 1) {
    tc_fence_after();
    if (CG2) tmem_dealloc_cg2(tmem_base, 512); else tmem_dealloc(tmem_base, 512);
  }
}
