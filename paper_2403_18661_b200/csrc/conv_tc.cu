// Host side of the tensor-core network path (fp16 weights and activations, fp32 accumulation): TMA tensor maps, per-layer launches, forward driver.
#include <map>
#include <string.h>

#include "conv_tc_kernel.cuh"
#include "conv_block_kernel.cuh"
#include "common.cuh"
#include "net_plan.h"
#include "stem.h"
#include <atomic>

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static bool encode_map(aframe_ctx* ctx, CUtensorMap* m, const void* ptr, int rank, const uint64_t* dims,
                       const uint64_t* strides_bytes /*rank-1*/, const uint32_t* box) {
  cuuint64_t gd[5], gs[4];
  cuuint32_t bx[5], es[5];
  for (int i = 0; i < rank; ++i) { gd[i] = dims[i]; bx[i] = box[i]; es[i] = 1; }
  for (int i = 0; i < rank - 1; ++i) gs[i] = strides_bytes[i];
  EncodeTiledFn fn = reinterpret_cast<EncodeTiledFn>(ctx->encode_tiled);
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, (cuuint32_t)rank, const_cast<void*>(ptr), gd, gs, bx, es,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(ctx->err, sizeof(ctx->err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return false;
  }
  return true;
}

#ifdef AFRAME_TC_CYCLES
// Experiments build only (nvcc -DAFRAME_TC_CYCLES; never part of the product library): per-role cycle counters of CTA 0,
// 32 slots per launch plan, handed out in build order and read back through aframe_experiment_tc_cycles.
static long long* g_tc_cycles = nullptr;
static int g_tc_cycles_next = 0;
static long long* tc_cycles_slot() {
  if (!g_tc_cycles) { cudaMalloc(&g_tc_cycles, sizeof(long long) * 32 * 256); cudaMemset(g_tc_cycles, 0, sizeof(long long) * 32 * 256); }
  return g_tc_cycles + 32 * (g_tc_cycles_next++ % 256);
}
AF_API int aframe_experiment_tc_cycles(long long* host_out /* [256][32] */) {
  if (!g_tc_cycles) return 0;
  cudaDeviceSynchronize();
  cudaMemcpy(host_out, g_tc_cycles, sizeof(long long) * 32 * 256, cudaMemcpyDeviceToHost);
  return g_tc_cycles_next;
}
#endif

struct TcLaunch {
  CUtensorMap tm_in, tm_w, tm_out, tm_res, tm_scw;
  TcConvParams p;
  int BN, grid, smem, device;
  bool head, cg2, halo;
  double macs = 0.0;   // multiply-accumulates the launch issues to the tensor cores (whole tiles, padding rows included)
};

// score[b] = (sum of the fused-head partials of window b) / T + bias   (deterministic: fixed summation order)
__global__ void head_finish_kernel(const float* __restrict__ part, int n_part, float inv_t, float bias, int64_t B,
                                   float* __restrict__ scores) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  float s = 0.f;
  for (int i = 0; i < n_part; ++i) s += part[b * n_part + i];
  scores[b] = s * inv_t + bias;
}

static int tile_t_box(int t_out) {
  if (t_out % 128 == 0) return 128;
  int tb = 1;
  while (tb < 128 && t_out % (tb * 2) == 0) tb *= 2;
  return tb;
}

// A conv layer runs on the tensor-core kernel if its channel counts tile into 64-wide K blocks / 64..256-wide N.
static bool tc_layer_ok(const LayerDesc& l, std::string& why) {
  if (l.c_in % 64) { why = "conv c_in not a multiple of 64"; return false; }
  if (!(l.c_out == 64 || l.c_out == 128 || l.c_out % 256 == 0)) { why = "conv c_out not 64, 128 or a multiple of 256"; return false; }
  if (!((l.k == 3 && l.pad == 1) || (l.k == 1 && l.pad == 0))) { why = "conv kernel/padding other than k3p1 / k1p0"; return false; }
  if (l.stride != 1 && l.stride != 2) { why = "conv stride other than 1 or 2"; return false; }
  if (l.t_in % l.stride) { why = "conv input length not divisible by its stride"; return false; }
  if (l.t_out * l.stride != l.t_in) { why = "conv output length != input length / stride"; return false; }
  if (tile_t_box(l.t_out) < 8) { why = "conv output length has no power-of-two factor >= 8"; return false; }
  return true;
}

aframe_status af_tc_check(aframe_ctx* ctx, aframe_weights* w) {
  w->tc_ok = false;
  const int n = (int)w->layers.size();
  if (!ctx->encode_tiled) { w->tc_reason = "cuTensorMapEncodeTiled entry point not found"; return AFRAME_OK; }
  if (n < 3 || w->layers[0].kind != 0 || w->layers[0].input_from != -1 || w->layers[1].kind != 1 ||
      w->layers[1].input_from != 0) { w->tc_reason = "table does not start with stem conv + max-pool"; return AFRAME_OK; }
  const LayerDesc& s = w->layers[0];
  const LayerDesc& q = w->layers[1];
  if (!(s.k == 7 && s.c_in == 2 && s.c_out == 64 && s.stride == 2 && s.pad == 3 && s.relu && s.residual_from < 0 &&
        q.k == 3 && q.stride == 2 && q.pad == 1)) { w->tc_reason = "stem is not conv(2->64,k7,s2,p3)+ReLU+maxpool(k3,s2,p1)"; return AFRAME_OK; }
  for (int i = 2; i < n; ++i) {
    const LayerDesc& l = w->layers[i];
    if (l.input_from == 0 || l.residual_from == 0 || l.input_from < 0) { w->tc_reason = "a layer reads the pre-pool stem output or the raw input"; return AFRAME_OK; }
    if (l.kind == 1) { w->tc_reason = "max-pool after the stem is not built on the bf16 path"; return AFRAME_OK; }
    if (l.kind == 0 && !tc_layer_ok(l, w->tc_reason)) return AFRAME_OK;
  }
  if (w->live_gn && (w->n_groups < 1 || w->n_groups > 32 || 64 % w->n_groups || (64 / w->n_groups) % 2)) {
    w->tc_reason = "true GroupNorm on the bf16 path needs an even number of stem channels per group"; return AFRAME_OK;
  }
  w->tc_ok = true;
  return AFRAME_OK;
}

// sc >= 0: layer sc is the 1x1 projection conv whose output is this layer's residual; it runs inside this launch as extra
// K blocks on its own input sc_in (res must then be null)
// ov != null (shared stages): the launch runs the layer on ONE long window of ov->t_out output rows (a stream, or a batch of
// short windows with zeroed separator rows) instead of nb windows of the table's length
// ov->e_nbp > 0 (packed edge batch, see TcConvParams::edge_nbp): 2 e_nbp short windows of e_P rows, one e_tbox-row box each
struct TcShapeOverride {
  int t_out; int zero_period, zero_valid, zero_origin;
  int e_nbp = 0, e_P = 0, e_tbox = 0, e_T = 0, e_head = 0, e_tail = 0;
  int64_t e_shift = 0, e_nb = 0;
  const af_act_t* e_stream = nullptr;
  int e_keep = 0;             // > 0: the slot's first / last e_keep rows must be valid (the next stage reads them in place); else e + 2

  // packed stages read their stage input in place: in_rows > 0: the (stream) launch's input tensor holds in_rows rows
  // (rows past them read as zero); e_Pin > 0: the edge launch's input slots hold e_Pin rows (the stage-input slots of the
  // entry conv and of the conv with the folded projection are only as long as those two layers reach)
  // (main: the layer's own input; sc: the input of the projection folded into it)
  int64_t in_rows = 0, in_rows_sc = 0;
  int e_Pin = 0, e_Pin_sc = 0;
  bool head_rows = false;     // with head = true: per-row head dot products into head_part (TcConvParams::head_rows)
  bool pair_plan = false;     // one shared-memory plan for every launch of the stage, so that two of them can share a launch
};
static bool build_launch(aframe_ctx* ctx, const aframe_weights* w, int li, const af_act_t* in,
                         const af_act_t* res, af_act_t* out, int64_t nb, bool head, float* head_part,
                         TcLaunch& L, int sc = -1, const af_act_t* sc_in = nullptr, const TcShapeOverride* ov = nullptr) {
  LayerDesc l = w->layers[li];
  const bool packed = ov && ov->e_nbp > 0;
  if (packed) { nb = 2 * ov->e_nbp; l.t_out = ov->e_P; l.t_in = ov->e_P * l.stride; }
  else if (ov) { nb = 1; l.t_out = ov->t_out; l.t_in = ov->t_out * l.stride; }
  // rows of the input tensor as the tensor map sees them (out-of-range rows are zero-filled by TMA)
  const int64_t in_rows = packed && ov->e_Pin > 0 ? ov->e_Pin : (ov && ov->in_rows > 0 ? ov->in_rows : l.t_in);
  const int BN = l.c_out >= 256 ? 256 : l.c_out;
  const bool cg2 = BN == 256;                                    // CTA pairs (cta_group::2) for the N = 256 layers
  const int T_box = packed ? ov->e_tbox : tile_t_box(l.t_out), B_box = 128 / T_box;
  const int P = l.stride;
  const bool has_res = res != nullptr;
  // resident weights + one halo box per tile (see TcConvParams): stride-1 k3 layers whose tiles stay inside a window
  bool halo = !head && !cg2 && l.k == 3 && l.stride == 1 && l.pad == 1 && T_box == 128 && BN == l.c_out && BN <= 128;
  {
    const uint64_t dims[4] = {(uint64_t)l.c_in, (uint64_t)P, (uint64_t)(in_rows / P), (uint64_t)nb};
    const uint64_t str[3] = {(uint64_t)l.c_in * 2, (uint64_t)P * l.c_in * 2, (uint64_t)in_rows * l.c_in * 2};
    const uint32_t box[4] = {64, 1, (uint32_t)(halo ? T_box + 2 : T_box), (uint32_t)B_box};
    if (!encode_map(ctx, &L.tm_in, in, 4, dims, str, box)) return false;
  }
  {
    const uint64_t dims[3] = {(uint64_t)l.c_in, (uint64_t)l.c_out, (uint64_t)l.k};
    const uint64_t str[2] = {(uint64_t)l.c_in * 2, (uint64_t)l.c_out * l.c_in * 2};
    const uint32_t box[3] = {64, (uint32_t)(cg2 ? BN / 2 : BN), 1};
    if (!encode_map(ctx, &L.tm_w, w->d_w16[li], 3, dims, str, box)) return false;
  }
  {
    const uint64_t dims[4] = {(uint64_t)l.c_out, 1, (uint64_t)l.t_out, (uint64_t)nb};
    const uint64_t str[3] = {(uint64_t)l.c_out * 2, (uint64_t)l.c_out * 2, (uint64_t)l.t_out * l.c_out * 2};
    const uint32_t box[4] = {64, 1, (uint32_t)T_box, (uint32_t)B_box};
    if (!encode_map(ctx, &L.tm_out, out, 4, dims, str, box)) return false;
    if (sc < 0 && !encode_map(ctx, &L.tm_res, res ? res : out, 4, dims, str, box)) return false;
  }
  L.tm_scw = L.tm_w;
  if (sc >= 0) {
    LayerDesc q = w->layers[sc];
    if (ov) { q.t_out = l.t_out; q.t_in = l.t_out * q.stride; }
    const int64_t sc_rows = packed && ov->e_Pin_sc > 0 ? ov->e_Pin_sc : (ov && ov->in_rows_sc > 0 ? ov->in_rows_sc : q.t_in);
    const uint64_t dims[4] = {(uint64_t)q.c_in, (uint64_t)q.stride, (uint64_t)(sc_rows / q.stride), (uint64_t)nb};
    const uint64_t str[3] = {(uint64_t)q.c_in * 2, (uint64_t)q.stride * q.c_in * 2, (uint64_t)sc_rows * q.c_in * 2};
    const uint32_t box[4] = {64, 1, (uint32_t)T_box, (uint32_t)B_box};
    if (!encode_map(ctx, &L.tm_res, sc_in, 4, dims, str, box)) return false;
    const uint64_t wd[3] = {(uint64_t)q.c_in, (uint64_t)q.c_out, 1};
    const uint64_t ws[2] = {(uint64_t)q.c_in * 2, (uint64_t)q.c_out * q.c_in * 2};
    const uint32_t wb[3] = {64, (uint32_t)(cg2 ? BN / 2 : BN), 1};
    if (!encode_map(ctx, &L.tm_scw, w->d_w16[sc], 3, wd, ws, wb)) return false;
  }
  TcConvParams& p = L.p;
  p.bias = sc >= 0 ? w->d_bias_sc[li] : w->d_bias[li];
  p.sc_kblocks = sc >= 0 ? w->layers[sc].c_in / 64 : 0;
  p.gn_part = nullptr; p.gn_unit = 64;
  p.zero_period = ov ? ov->zero_period : 0; p.zero_valid = ov ? ov->zero_valid : 0; p.zero_origin = ov ? ov->zero_origin : 0;
  p.taps = l.k; p.pad = l.pad; p.P = P;
  for (int d = 0; d < 3; ++d) {
    const int sft = d - l.pad;
    const int toff = sft >= 0 ? sft / P : -((-sft + P - 1) / P);
    p.tap_toff[d] = toff; p.tap_par[d] = sft - toff * P;
  }
  p.kblocks = l.c_in / 64;
  p.n_tiles = l.c_out / BN;
  p.T_box = T_box; p.B_box = B_box;
  p.t_blks = packed ? 1 : l.t_out / T_box;
  p.a_bytes = T_box * B_box * 128;
  p.edge_nbp = packed ? ov->e_nbp : 0;
  p.edge_blks_half = packed ? (int)((ov->e_nb + B_box - 1) / B_box) : 0;
  p.edge_t0_tail = packed ? ov->e_P - T_box : 0;
  // ... and where a tail box starts in the slots it READS (in output-row units of this layer): slots of the previous layer's
  // output are as long as this layer's; stage-input slots (e_Pin rows at the previous stage's resolution) are shorter
  p.edge_t0_tail_in = packed ? (int)(in_rows / P) - T_box : 0;
  p.edge_t0_tail_sc = packed && sc >= 0 ? (int)((ov->e_Pin_sc > 0 ? ov->e_Pin_sc : w->layers[sc].stride * ov->e_P) / w->layers[sc].stride) - T_box : 0;
  p.edge_T = packed ? ov->e_T : 0; p.edge_P = packed ? ov->e_P : 0;
  p.edge_head = packed ? ov->e_head : 0; p.edge_tail = packed ? ov->e_tail : 0;
  p.edge_shift = packed ? ov->e_shift : 0;
  p.edge_stream = packed ? reinterpret_cast<const uint4*>(ov->e_stream) : nullptr;
  // the two stream rows next to a slot's edge rows, as far as the box does not hold them (the store warp copies those)
  p.edge_out = packed && ov->e_stream ? reinterpret_cast<uint4*>(out) : nullptr;
  p.cpy_t0_head = p.cpy_n_head = p.cpy_t0_tail = p.cpy_n_tail = 0;
  if (p.edge_out) {
    const int need_h = ov->e_keep > 0 ? ov->e_keep : ov->e_head + 2, need_t = ov->e_keep > 0 ? ov->e_keep : ov->e_tail + 2;
    p.cpy_t0_head = ov->e_head > T_box ? ov->e_head : T_box;
    p.cpy_n_head = need_h - p.cpy_t0_head;
    p.cpy_t0_tail = ov->e_T - need_t;
    p.cpy_n_tail = need_t - (ov->e_tail > T_box ? ov->e_tail : T_box);
    if (p.cpy_n_head < 0) p.cpy_n_head = 0;
    if (p.cpy_n_tail < 0) p.cpy_n_tail = 0;
  }
  const int64_t b_blks = packed ? 2 * ((ov->e_nb + B_box - 1) / B_box) : (nb + B_box - 1) / B_box;
  const int64_t m_tiles = b_blks * p.t_blks;
  p.num_tiles = (int)((cg2 ? (m_tiles + 1) / 2 : m_tiles) * p.n_tiles);
  L.macs = (double)(cg2 ? 2 * ((m_tiles + 1) / 2) : m_tiles) * 128.0 * l.c_out * 64.0 * (l.k * (l.c_in / 64) + (sc >= 0 ? w->layers[sc].c_in / 64 : 0));
  p.div_n = tc_fastdiv((uint32_t)p.n_tiles);
  p.div_t = tc_fastdiv((uint32_t)p.t_blks);
  p.div_tbox = tc_fastdiv((uint32_t)T_box);
  // true GroupNorm (NEXT-2): the conv stores its plain output; norm, residual and ReLU follow in af_launch_gn_bf16
  p.relu = w->live_gn ? 0 : l.relu; p.has_res = res != nullptr;
  p.c_out = l.c_out;
  p.head_w = head ? w->d_head_w : nullptr;
  p.head_part = head ? head_part : nullptr;
  p.head_slabs = l.t_out / 32;
  p.head_rows = (head && ov && ov->head_rows) ? 1 : 0; p.head_row_stride = l.t_out;
  p.head_rows_total = (long long)l.t_out * nb;
  p.nb = packed ? ov->e_nb : nb;
#ifdef AFRAME_TC_CYCLES
  p.dbg_out = tc_cycles_slot();
#endif
  // shared-memory plan (227 KB per CTA): main-loop ring depth vs epilogue staging / residual prefetch buffers
  // (two epilogue groups: EG * nbuf staging buffers of 16 KB; a residual tile is prefetched pf chunks ahead into the
  //  buffer its chunk's output is staged in)
  const bool r = p.has_res;
  if (cg2 && !head && BN == 256 && ov && ov->pair_plan) { p.stages = 5; p.nbuf = 2; p.pf = 1; }
  else if (cg2 && head)       { p.stages = 5; p.nbuf = 1; p.pf = 0; }
  else if (cg2 && l.k * p.kblocks < 12) { p.stages = 5; p.nbuf = 2; p.pf = r ? 1 : 0; }   // short K: the epilogue is the critical path
  else if (cg2)               { p.stages = r ? 5 : 6; p.nbuf = r ? 2 : 1; p.pf = r ? 1 : 0; }
  else if (BN == 256)         { p.stages = 3; p.nbuf = 2; p.pf = r ? 1 : 0; }
  else if (halo && BN == 128 && sc >= 0) { p.stages = 3; p.nbuf = 1; p.pf = 0; }   // 96 + 16 KB of weights + 3 x 17 KB + 2 x 16 KB
  else if (halo && BN == 128) { p.stages = 3; p.nbuf = 2; p.pf = r ? 1 : 0; }   // 96 KB of weights + 3 x 17 KB + 4 x 16 KB
  else if (halo)              { p.stages = r ? 6 : 8; p.nbuf = r ? 3 : 2; p.pf = r ? 1 : 0; }
  else if (BN == 128)         { p.stages = r ? 4 : 5; p.nbuf = r ? 3 : 2; p.pf = r ? 1 : 0; }
  else                        { p.stages = r ? 5 : 6; p.nbuf = r ? 3 : 2; p.pf = r ? 1 : 0; }
  p.w_bytes = halo ? (l.k * p.kblocks + p.sc_kblocks) * BN * 128 : 0;
  p.stage_bytes = halo ? TcCfg<64>::HALO_A_BYTES : 0;     // one stage = one 64-channel block

  L.BN = BN;
  L.device = ctx->device;
  L.head = head;
  L.cg2 = cg2;
  L.halo = halo;
  L.smem = halo ? (BN == 128 ? TcCfg<128>::smem_halo(p.stages, p.nbuf, l.k, p.kblocks) : TcCfg<64>::smem_halo(p.stages, p.nbuf, l.k, p.kblocks)) + p.sc_kblocks * BN * 128
         : cg2 ? TcCfg<256, true>::smem(p.stages, p.nbuf, head) : (BN == 128 ? TcCfg<128>::smem(p.stages, p.nbuf, head)
                                                                            : TcCfg<64>::smem(p.stages, p.nbuf, head));
  if (cg2) L.grid = 2 * (p.num_tiles < ctx->n_sms / 2 ? p.num_tiles : ctx->n_sms / 2);
  else L.grid = p.num_tiles < ctx->n_sms ? p.num_tiles : ctx->n_sms;
  return true;
}

template <int BN, bool HEAD, bool CG2, bool HALO = false> static cudaError_t launch_bn(const TcLaunch& L, cudaStream_t s,
                                                                                   const TcLaunch* second = nullptr) {
  static std::atomic<uint64_t> attr_done{0};          // bit d: the attribute is set on device d (it is per device)
  auto kern = conv_tc_kernel<BN, HEAD, CG2, HALO>;
  const uint64_t bit = 1ull << (L.device & 63);
  if (!(attr_done.load(std::memory_order_acquire) & bit)) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448);
    if (e != cudaSuccess) return e;
    attr_done.fetch_or(bit, std::memory_order_release);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)L.grid);
  cfg.blockDim = dim3((unsigned)TcCfg<BN, CG2>::THREADS);
  cfg.dynamicSmemBytes = (size_t)L.smem;
  cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = CG2 ? 2 : 1; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // the kernel orders itself with griddepcontrol.wait
  at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 2;
  const TcLaunch& L1 = second ? *second : L;        // second problem of the launch (conv_tc_kernel), or none
  TcConvParams p1 = L1.p;
  if (!second) p1.num_tiles = 0;
  return cudaLaunchKernelEx(&cfg, kern, L.tm_in, L.tm_w, L.tm_out, L.tm_res, L.tm_scw, L.p, L1.tm_in, L1.tm_w, L1.tm_out, L1.tm_res,
                            L1.tm_scw, p1);
}

// second != null: both problems in one launch (only the CTA-pair N = 256 storing variant is paired, see can_pair below)
static cudaError_t launch_conv(const TcLaunch& L, cudaStream_t s, const TcLaunch* second = nullptr) {
  if (L.cg2) return L.head ? launch_bn<256, true, true>(L, s) : launch_bn<256, false, true>(L, s, second);
  if (L.halo) return L.BN == 128 ? launch_bn<128, false, false, true>(L, s) : launch_bn<64, false, false, true>(L, s);
  return L.BN == 128 ? launch_bn<128, false, false>(L, s) : launch_bn<64, false, false>(L, s);
}

// fused basic block (conv_block_kernel): layers a (conv) and b (conv + residual from a's input)
struct TcBlockLaunch {
  CUtensorMap tm_x, tm_wa, tm_wb, tm_out;
  TcBlockParams p;
  int grid = 0, smem = 0, device = 0;
  double macs = 0.0;   // as TcLaunch::macs (two convs, 128-row MMAs per 126-row tile)
};

// Layer i is the first conv of a basic block the fused kernel can run: 64 -> 64 -> 64 channels, k3 s1 p1, ReLU after each,
// the second conv adds the block input, and nothing else reads the intermediate tensor.
static int fusable_block(const std::vector<LayerDesc>& layers, int i) {
  const int n = (int)layers.size();
  if (i < 2 || i + 1 >= n) return -1;
  const LayerDesc& a = layers[i];
  const LayerDesc& b = layers[i + 1];
  auto conv3 = [](const LayerDesc& l) { return l.kind == 0 && l.k == 3 && l.stride == 1 && l.pad == 1 && l.relu && l.c_in == 64 && l.c_out == 64; };
  if (!conv3(a) || !conv3(b) || a.residual_from >= 0 || b.input_from != i || b.residual_from != a.input_from) return -1;
  for (int j = 0; j < n; ++j)
    if (j != i + 1 && (layers[j].input_from == i || layers[j].residual_from == i)) return -1;
  return i + 1;
}
static int fusable_block(const aframe_weights* w, int i) { return fusable_block(w->layers, i); }

// Layer i adds the output of a 1x1 projection conv of the same width (aframe_weights_load then keeps the sum of the two
// folded biases in d_bias_sc[i], and the projection can run inside layer i as extra K blocks)
static bool has_projection_residual(const std::vector<LayerDesc>& layers, int i) {
  const LayerDesc& l = layers[i];
  if (l.kind != 0 || l.residual_from < 0) return false;
  const LayerDesc& r = layers[l.residual_from];
  return r.kind == 0 && r.k == 1 && r.c_out == l.c_out;
}

// row_shift > 0: x is the stem of the whole stream (shared stem): window b starts row_shift rows after window b - 1, and
// edge holds every window's own rows 0, 1, T - 1
static bool build_block_launch(aframe_ctx* ctx, const aframe_weights* w, int ia, int ib, const af_act_t* x,
                               af_act_t* out, int64_t nb, TcBlockLaunch& L, int64_t row_shift = 0,
                               const af_act_t* edge = nullptr, int T_override = 0, int zero_period = 0, int zero_valid = 0) {
  const LayerDesc& a = w->layers[ia];
  const int T = T_override > 0 ? T_override : a.t_out;
  const uint64_t dims[3] = {64, (uint64_t)T, (uint64_t)nb};
  const uint64_t str[2] = {128, (uint64_t)T * 128};
  const uint64_t str_x[2] = {128, (uint64_t)(row_shift > 0 ? row_shift : T) * 128};
  const uint32_t box_x[3] = {64, 130, 1}, box_o[3] = {64, TCB_ROWS, 1}, box_w[3] = {64, 64, 1};
  const uint64_t wd[3] = {64, 64, 3};
  const uint64_t ws[2] = {128, 64 * 128};
  if (!encode_map(ctx, &L.tm_x, x, 3, dims, str_x, box_x) || !encode_map(ctx, &L.tm_out, out, 3, dims, str, box_o) ||
      !encode_map(ctx, &L.tm_wa, w->d_w16[ia], 3, wd, ws, box_w) || !encode_map(ctx, &L.tm_wb, w->d_w16[ib], 3, wd, ws, box_w))
    return false;
  TcBlockParams& p = L.p;
  p.bias_a = w->d_bias[ia]; p.bias_b = w->d_bias[ib];
  p.T = T;
  p.tiles_per_win = (T + TCB_ROWS - 1) / TCB_ROWS;
  p.num_tiles = (int)(nb * p.tiles_per_win);
  p.div_tw = tc_fastdiv((uint32_t)p.tiles_per_win);
  p.nx = 6; p.ny = 2; p.no = 1;
  p.edge = row_shift > 0 ? edge : nullptr;
  p.zero_period = zero_period; p.zero_valid = zero_valid;
  p.reverse = 0;
#ifdef AFRAME_TC_CYCLES
  p.dbg_out = tc_cycles_slot();
#endif
  L.smem = tcb_smem(p.nx, p.ny, p.no);
  L.device = ctx->device;
  L.grid = p.num_tiles < ctx->n_sms ? p.num_tiles : ctx->n_sms;
  L.macs = 2.0 * p.num_tiles * 128.0 * 64.0 * 192.0;
  return true;
}

static cudaError_t launch_block(const TcBlockLaunch& L, cudaStream_t s) {
  static std::atomic<uint64_t> attr_done{0};
  const uint64_t bit = 1ull << (L.device & 63);
  if (!(attr_done.load(std::memory_order_acquire) & bit)) {
    cudaError_t e = cudaFuncSetAttribute(conv_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448);
    if (e != cudaSuccess) return e;
    attr_done.fetch_or(bit, std::memory_order_release);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)L.grid);
  cfg.blockDim = dim3(576);
  cfg.dynamicSmemBytes = (size_t)L.smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, conv_block_kernel, L.tm_x, L.tm_wa, L.tm_wb, L.tm_out, L.p);
}

// ---- shared first stage -----------------------------------------------------------------------------------------
// Windows spaced row_shift rows apart in the stem's stream overlap, and so do the outputs of every stride-1 'same' conv
// that follows: a row is identical in all windows that hold it EXCEPT in the windows where it lies within reach of that
// window's zero padding (each conv widens this edge by one row per side).  The fused blocks of the 64-channel stage
// therefore run (1) once over the whole stream and (2) over a batch of 2 short windows per window -- its first and last
// S1_ROWS rows, with the true edge rows of the previous block -- which yields the edge rows exactly; s1_stitch_kernel
// then writes the per-window tensor the next stage reads.  Same kernel, same per-row arithmetic: bit-identical results.
constexpr int SH_SPARE_SLOTS = 32;          // packed edge batch: spare slots after each half (the last box of a half may overhang)
constexpr int S1_ROWS = 16;                 // rows of a short window (needs 2 K + 4 <= S1_ROWS - 2 for K blocks)
constexpr int S1_PERIOD = S1_ROWS + 2;      // + 2 separator rows (zero input, y1 forced to zero)

// X[m][r] for short window m = 2 b + tail, r < S1_PERIOD: window row t = r (head) or T - S1_ROWS + r (tail), taken from
// the previous block's edge results where the row is an edge row there, else from the previous block's stream.
__global__ void s1_gather_kernel(uint4* __restrict__ X, const uint4* __restrict__ S_prev, const uint4* __restrict__ Y_prev,
                                 const uint4* __restrict__ E0, int64_t nb, int T, int64_t row_shift, int c_head, int c_tail) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * nb * S1_PERIOD * 8) return;
  const int j = (int)(i & 7);
  const int64_t mr = i >> 3;
  const int r = (int)(mr % S1_PERIOD);
  const int64_t m = mr / S1_PERIOD, b = m >> 1;
  const bool tail = (m & 1) != 0;
  uint4 v = make_uint4(0u, 0u, 0u, 0u);
  if (r < S1_ROWS) {
    const int t = tail ? T - S1_ROWS + r : r;
    const bool from_edge = tail ? (t >= T - c_tail) : (t < c_head);
    if (from_edge) v = E0 ? E0[(b * 3 + (tail ? 2 : t)) * 8 + j] : Y_prev[(m * S1_PERIOD + r) * 8 + j];
    else v = S_prev[(b * row_shift + t) * 8 + j];
  }
  X[i] = v;
}

// out[b][t] = the last block's edge result where t is an edge row of window b, else its stream row
__global__ void s1_stitch_kernel(uint4* __restrict__ out, const uint4* __restrict__ S, const uint4* __restrict__ Y, int64_t nb,
                                 int T, int64_t row_shift, int c_head, int c_tail) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nb * T * 8) return;
  const int j = (int)(i & 7);
  const int64_t bt = i >> 3;
  const int t = (int)(bt % T);
  const int64_t b = bt / T;
  uint4 v;
  if (t < c_head) v = Y[((2 * b) * S1_PERIOD + t) * 8 + j];
  else if (t >= T - c_tail) v = Y[((2 * b + 1) * S1_PERIOD + (t - (T - S1_ROWS))) * 8 + j];
  else v = S[(b * row_shift + t) * 8 + j];
  out[i] = v;
}

// ---- shared second stage ---------------------------------------------------------------------------------------------
// The stage that follows (stride-2 entry conv + 1x1 projection + stride-1 convs) is shift-equivariant in the same way at
// half the row spacing.  Its layers run unchanged (conv_tc_kernel) on (1) the stream, as one long window, and (2) a batch
// of two short windows per window -- the first / last S2_ROWS output rows, i.e. 2 S2_ROWS input rows -- separated by zeroed
// rows (TcConvParams::zero_period), then s2_stitch_kernel writes the per-window tensor the next stage reads.
// A stage's short windows hold `rows` output rows (the smallest count that keeps every edge row out of reach of the short
// window's artificial end: edge rows + convs after the entry conv) and repeat every `period` = rows + 2 rows (2 separators).

// Input of a stage's short windows at the previous stage's resolution: [short windows][2 S2_PERIOD rows][pieces * 8 ch];
// local row r < 2 S2_ROWS is window row r (head) or Tp - 2 S2_ROWS + r (tail), taken from the previous stage's edge batch
// (period src_period, src_rows data rows per short window) where it is an edge row there (rows < c_head or >= Tp - c_tail),
// else from the previous stage's stream; the other rows are zero.
__global__ void sh_gather_kernel(uint4* __restrict__ X, const uint4* __restrict__ S, const uint4* __restrict__ Y, int64_t nb,
                                 int64_t n_short /* short windows incl. padding */, int Tp, int pieces, int64_t row_shift,
                                 int src_period, int src_rows, int c_head, int c_tail, int64_t copy_rows, int64_t valid_rows,
                                 int rows, int period, int64_t edge_rows_in /* rows of the short-window part of X */) {
  // X = [copy_rows rows: the previous stage's stream (its first valid_rows rows; the last 4 rows zero: they are the first short
  //      window's padding at this resolution) | n_short short windows of 2 S2_PERIOD rows]
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (copy_rows + edge_rows_in) * pieces) return;
  const int j = (int)(i % pieces);
  const int64_t row = i / pieces;
  uint4 v = make_uint4(0u, 0u, 0u, 0u);
  if (row < copy_rows) {
    if (row < valid_rows && row < copy_rows - 4) v = S[row * pieces + j];
    X[i] = v;
    return;
  }
  const int64_t mr = row - copy_rows;
  const int r = (int)(mr % (2 * period));
  const int64_t m = mr / (2 * period), b = m >> 1;
  const bool tail = (m & 1) != 0;
  if (r < 2 * rows && b < nb && m < n_short) {
    const int t = tail ? Tp - 2 * rows + r : r;
    if (!tail && t < c_head) v = Y[(m * src_period + t) * pieces + j];
    else if (tail && t >= Tp - c_tail) v = Y[(m * src_period + (t - (Tp - src_rows))) * pieces + j];
    else v = S[(b * row_shift + t) * pieces + j];
  }
  X[i] = v;
}

// Packed edge batch (stages on the CTA-pair path, see TcConvParams::edge_nbp): X = [copy_rows rows: the previous stage's stream |
// nbp slots of P2 rows: the first P2 rows of every window | nbp slots: the last P2 rows of every window], each row taken from
// the previous stage's edge batch where it is an edge row there, else from its stream.
__global__ void shp_gather_kernel(uint4* __restrict__ X, const uint4* __restrict__ S, const uint4* __restrict__ Y, int64_t nb,
                                  int64_t nbp, int Tp, int pieces, int64_t row_shift, int64_t src_stride, int64_t src_tail0,
                                  int src_trow, int c_head, int c_tail, int64_t copy_rows, int64_t valid_rows, int P2) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (copy_rows + 2 * nbp * P2) * pieces) return;
  const int j = (int)(i % pieces);
  const int64_t row = i / pieces;
  uint4 v = make_uint4(0u, 0u, 0u, 0u);
  if (row < copy_rows) {
    if (row < valid_rows) v = S[row * pieces + j];
    X[i] = v;
    return;
  }
  const int64_t mr = row - copy_rows;
  const int r = (int)(mr % P2);
  const int64_t m = mr / P2;
  const bool tail = m >= nbp;
  const int64_t b = tail ? m - nbp : m;
  if (b < nb) {
    const int t = tail ? Tp - P2 + r : r;
    if (!tail && t < c_head) v = Y[(b * src_stride + t) * pieces + j];
    else if (tail && t >= Tp - c_tail) v = Y[(src_tail0 + b * src_stride + (t - src_trow)) * pieces + j];
    else v = S[(b * row_shift + t) * pieces + j];
  }
  X[i] = v;
}

// out[b][t][C]: edge result where t is an edge row of window b (t < c_head or t >= T2 - c_tail), else the stream row
// (edge batch addressing, both layouts: window b's first rows start at row b * e_stride, its last rows at e_tail0 + b * e_stride,
//  where local row 0 is window row e_trow)
__global__ void s2_stitch_kernel(uint4* __restrict__ out, const uint4* __restrict__ S, const uint4* __restrict__ Y, int64_t nb,
                                 int T2, int pieces /* C / 8 */, int64_t row_shift, int c_head, int c_tail, int64_t e_stride,
                                 int64_t e_tail0, int e_trow) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nb * T2 * pieces) return;
  const int j = (int)(i % pieces);
  const int64_t bt = i / pieces;
  const int t = (int)(bt % T2);
  const int64_t b = bt / T2;
  uint4 v;
  if (t < c_head) v = Y[(b * e_stride + t) * pieces + j];
  else if (t >= T2 - c_tail) v = Y[(e_tail0 + b * e_stride + (t - e_trow)) * pieces + j];
  else v = S[(b * row_shift + t) * pieces + j];
  out[i] = v;
}

// Fused-head partials for a stage that ran in shared form: the same numbers, summed in the same order, as the HEAD variant of
// conv_tc_kernel emits from its epilogue.  The stage's last conv stores no activation (TcConvParams::head_rows): its epilogue
// emits each row's dot product with the head weights per head unit (the channels one epilogue thread holds), Rs over the
// stream and Re over the edge batch; here one warp = one 32-row slab of one window x one unit, lane = row of the slab, and
// the 32 values are summed in the order the fused head uses.  head_finish_kernel then sums the partials as usual.
__global__ void __launch_bounds__(256)
sh_head_rows_kernel(const float* __restrict__ Rs, int64_t rows_s, const float* __restrict__ Re, int64_t rows_e,
                    float* __restrict__ head_part, int64_t nb, int T, int chunks, int64_t row_shift, int c_head, int c_tail,
                    int64_t e_stride, int64_t e_tail0, int e_trow) {
  // one warp per (window, slab), lane = row; the head units are walked in a loop (one 32-bit division per warp instead of
  // three 64-bit ones per (window, slab, unit): the first version was bound by them)
  const int lane = threadIdx.x & 31;
  const int slabs = T / 32;
  const unsigned wi = blockIdx.x * 8u + (threadIdx.x >> 5);
  if (wi >= (unsigned)(nb * slabs)) return;
  const unsigned b = wi / (unsigned)slabs;
  const int slab = (int)(wi - b * (unsigned)slabs);
  const int t = slab * 32 + lane;
  const float* src;
  int64_t unit_stride;
  if (t < c_head) { src = Re + (int64_t)b * e_stride + t; unit_stride = rows_e; }
  else if (t >= T - c_tail) { src = Re + e_tail0 + (int64_t)b * e_stride + (t - e_trow); unit_stride = rows_e; }
  else { src = Rs + (int64_t)b * row_shift + t; unit_stride = rows_s; }
  float* dst = head_part + ((int64_t)b * slabs + slab) * chunks;
  for (int c0 = 0; c0 < chunks; c0 += 4) {         // four units in flight
    float v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = c0 + k < chunks ? __ldg(src + (c0 + k) * unit_stride) : 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      float sum = v[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
      if (lane == 0 && c0 + k < chunks) dst[c0 + k] = sum;
    }
  }
}

struct TcPlanCache {
  const aframe_weights* w = nullptr;
  void* base = nullptr;
  int64_t nb = 0;
  size_t slot_bytes = 0;
  std::vector<TcLaunch> launches;   // indexed by layer
  std::vector<TcBlockLaunch> blocks;  // indexed by the block's SECOND layer
  std::vector<int> fused_with;        // per layer: index of the partner layer if the pair runs fused, else -1
  int64_t win_stride = 0;             // input window spacing the plans were built for (shared stem)
  bool shared_stem = false;           // stem of the whole stream + edge rows instead of one stem per window
  int s1_blocks = 0;                  // > 0: the first s1_blocks fused blocks run in shared form (see s1_gather_kernel)
  std::vector<TcBlockLaunch> s1_stream, s1_edge;
  struct SharedStagePlan {
    std::vector<int> layers;          // these layers (entry conv, then the stride-1 convs) run in shared form
    std::vector<TcLaunch> stream, edge;   // parallel to layers
    int T = 0, C = 0, C_in = 0, head = 0, tail = 0;   // output rows / channels, input channels, edge rows per window
    int rows = 0, period = 0;         // short window: data rows, data + separator rows
    int64_t shift = 0;                // rows between consecutive windows
    bool packed = false;              // packed edge batch: separate stream / edge launches per layer (TcConvParams::edge_nbp)
    int P = 0;                        // packed: rows per short-window slot
    int64_t nbp = 0;                  // packed: slots per half (windows rounded up to whole boxes)
    int64_t e_stride = 0, e_tail0 = 0; int e_trow = 0;   // edge-batch addressing of the stage's output (see s2_stitch_kernel)
  };
  std::vector<SharedStagePlan> sh;    // the stages after the first that run in shared form, in order
  bool sh_head = false;               // the last shared stage feeds the fused head: sh_head_partial_kernel instead of a stitch
  bool sh_head_rows = false;          // ... and its last conv emits per-row head dot products (sh_head_rows_kernel)
  std::vector<int> sc_of;             // per layer: the projection-shortcut conv that runs inside it (else -1)
  std::vector<char> skip;             // per layer: runs inside another launch
};
// the launch plans live in the context (ctx->tc_cache), so contexts never share mutable state
void af_tc_forget(aframe_ctx* ctx) {
  delete static_cast<std::vector<TcPlanCache>*>(ctx->tc_cache);
  ctx->tc_cache = nullptr;
}

// Windows per internal launch sequence.  Measured on B200: every layer launch carries ~12 us of launch gap, prologue
// (TMEM/barriers/first loads from HBM) and drain, so large chunks win (592: 869, 1184: 922, 4096: 994 TFLOP/s); the three
// live activation tensors leave the 126 MB L2 from ~300 windows on anyway.
static int64_t tc_chunk_windows() { return 8192; }

// Number of leading fused 64-channel blocks that form a chain on the pooled stem output (layers 2,3 | 4,5 | ...): the
// blocks the shared first stage can take over.
static int s1_chain_blocks(const std::vector<LayerDesc>& layers) {
  const int n = (int)layers.size();
  int k = 0, prev = 1;
  for (int i = 2; i + 1 < n && k < 5; i += 2) {
    if (fusable_block(layers, i) != i + 1 || layers[i].input_from != prev || layers[i + 1].residual_from != prev) break;
    bool other = false;                              // the block input must have no reader outside the block
    for (int j = 2; j < n; ++j)
      if (j != i && j != i + 1 && (layers[j].input_from == prev || layers[j].residual_from == prev)) other = true;
    if (other) break;
    prev = i + 1;
    ++k;
  }
  return k;
}

// Layers of the stage after the shared first stage, if it has the form the shared second stage handles: entry conv k3 s2
// (i0), projection k1 s2 (i0 + 1, folded into i0 + 2), then stride-1 k3 convs in basic blocks, all with the same width.
// Returns the layers that launch, in order (i0, i0 + 2, i0 + 3, ...); empty if the pattern does not match.
static std::vector<int> s2_chain_layers(const std::vector<LayerDesc>& layers, int i0) {
  std::vector<int> out;
  const int n = (int)layers.size();
  if (i0 + 2 >= n - 1) return out;
  const int prev = i0 - 1;
  const LayerDesc& e = layers[i0];
  const LayerDesc& q = layers[i0 + 1];
  const LayerDesc& f = layers[i0 + 2];
  auto conv3 = [&](const LayerDesc& l, int stride) { return l.kind == 0 && l.k == 3 && l.stride == stride && l.pad == 1 && l.relu && l.c_out == e.c_out; };
  if (!conv3(e, 2) || e.input_from != prev || e.residual_from >= 0) return out;
  if (!(q.kind == 0 && q.k == 1 && q.stride == 2 && q.pad == 0 && !q.relu && q.input_from == prev && q.residual_from < 0 && q.c_out == e.c_out)) return out;
  if (!conv3(f, 1) || f.input_from != i0 || f.residual_from != i0 + 1 || !has_projection_residual(layers, i0 + 2)) return out;
  for (int j = 2; j < n; ++j)                     // the first stage's output feeds only the entry conv and the projection
    if (j != i0 && j != i0 + 1 && (layers[j].input_from == prev || layers[j].residual_from == prev)) return out;
  out.push_back(i0); out.push_back(i0 + 2);
  int blk_in = i0 + 2;
  for (int j = i0 + 3; j + 1 < n - 1; j += 2) {
    const LayerDesc& a = layers[j];
    const LayerDesc& b = layers[j + 1];
    if (!conv3(a, 1) || !conv3(b, 1) || a.input_from != blk_in || a.residual_from >= 0 || b.input_from != j || b.residual_from != blk_in) break;
    out.push_back(j); out.push_back(j + 1);
    blk_in = j + 1;
  }
  // every tensor inside the chain is read only inside the chain (the last one is stitched for whoever reads it)
  const int last = out.back();
  for (int j = 2; j < n; ++j) {
    if (j >= i0 && j <= last) continue;
    const int a = layers[j].input_from, r = layers[j].residual_from;
    if ((a >= i0 && a < last) || (r >= i0 && r < last)) { out.clear(); return out; }
  }
  return out;
}


// ---- the shared-stage plan: host arithmetic only (no CUDA call), so that it can be unit-tested without a device --------
constexpr int TC_MAX_SHARED_STAGES = 3;
struct SharedStage {
  std::vector<int> list;            // layers that launch, entry conv first
  int i0 = 0, T = 0, C = 0, C_in = 0, head = 0, tail = 0;
  int rows = 0, period = 0;         // short window: data rows, data + 2 separator rows
  int64_t shift = 0;                // rows between consecutive windows at this stage's resolution
  int64_t rows_stream = 0, rows_edge = 0;
  size_t stream_bytes = 0, edge_bytes = 0, x_bytes = 0, off = 0;
  // packed edge batch (stages whose layers run on the CTA-pair path): P rows per short-window slot, per launched layer the
  // edge rows of its output at the window's start / end and the rows its box computes
  bool packed = false;
  int P = 0, P_in = 0;              // rows per slot of the layers' outputs / of the gathered stage input
  bool in_place = false;            // the stage reads the previous (packed) stage's last-layer slots in place: no gather
  int keep = 0;                     // > 0: the next stage does; the last layer's slots hold `keep` valid rows at each end
  std::vector<int> e_head, e_tail, tbox;
};
struct SharedPlan {
  int fuse = -1;                    // conv whose epilogue runs the head (else -1)
  int s1_k = 0;                     // fused 64-channel blocks on the pooled stem output
  bool s1_on = false;               // ... that run in shared form
  bool sh_head_on = false;          // the last shared stage ends in the fused head
  std::vector<SharedStage> stages;  // the shared stages after the first
};
static int64_t tc_up128(int64_t v) { return (v + 127) / 128 * 128; }

// layers: the table with t_in / t_out filled; sB: window spacing in samples; chunk: windows per launch sequence
static SharedPlan tc_plan_shared(const std::vector<LayerDesc>& layers, bool live_gn, int64_t sB, int64_t chunk) {
  SharedPlan pl;
  const int n = (int)layers.size();
  {
    // fused head: the conv feeding the head (and nothing else) pools + dots in its epilogue and stores nothing
    const LayerDesc& h = layers[n - 1];
    const int src = h.input_from;
    bool only_consumer = src >= 2 && layers[src].kind == 0;
    for (int i = 0; only_consumer && i < n - 1; ++i)
      if (layers[i].input_from == src || layers[i].residual_from == src) only_consumer = false;
    if (only_consumer && layers[src].c_out % 256 == 0 && layers[src].c_out <= 512 && tile_t_box(layers[src].t_out) % 32 == 0 && !live_gn)
      pl.fuse = src;
  }
  pl.s1_k = s1_chain_blocks(layers);
  pl.s1_on = pl.s1_k > 0 && sB % 4 == 0 && sB < layers[0].t_in && chunk >= 2 && !live_gn && layers[1].t_out >= 2 * S1_ROWS;
  if (!pl.s1_on) return pl;
  std::vector<SharedStage>& shs = pl.stages;
  int i0 = 2 + 2 * pl.s1_k, Tp = layers[1].t_out, hp = 2 * pl.s1_k + 2, tp = 2 * pl.s1_k + 1;
  int64_t shift_p = sB / 4;
  while ((int)shs.size() < TC_MAX_SHARED_STAGES && shift_p % 2 == 0 && !pl.sh_head_on) {
    SharedStage g;
    g.list = s2_chain_layers(layers, i0);
    if (g.list.empty()) break;
    if (pl.fuse >= i0 && pl.fuse <= g.list.back()) {
      // the stage that ends in the fused head: its last conv emits per-row head dot products (sh_head_rows_kernel);
      // needs whole 32-row slabs and the head as the only reader
      if (pl.fuse != g.list.back() || layers[pl.fuse].t_out % 32 != 0) break;
      pl.sh_head_on = true;
    }
    const int n2 = (int)g.list.size() - 1;
    g.i0 = i0; g.T = layers[i0].t_out; g.C = layers[i0].c_out; g.C_in = layers[i0].c_in;
    g.shift = shift_p / 2;
    g.head = hp / 2 + 1 + n2;                                   // rows within reach of the window's zero padding ...
    g.tail = g.T - (Tp - tp) / 2 + n2;                          // ... at the start and at the end of the stage's output
    const int src_rows = shs.empty() ? S1_ROWS : shs.back().rows;
    g.rows = g.head + n2 > g.tail + n2 + 1 ? g.head + n2 : g.tail + n2 + 1;
    g.period = g.rows + 2;
    // (head + tail <= T: a row taken from the window's first rows must be out of reach of the padding at its END, which the
    //  short window at the start does not see, and vice versa; short windows at both ends of short windows would overlap)
    const bool fits = g.T >= g.rows && Tp >= 2 * g.rows && Tp == 2 * g.T && hp <= src_rows - 2 && tp <= src_rows - 2 &&
                      g.C % 64 == 0 && g.C_in % 64 == 0 && g.head + g.tail <= g.T;
    if (!fits) { pl.sh_head_on = false; break; }
    g.rows_stream = tc_up128((chunk - 1) * g.shift + g.T);
    g.rows_edge = tc_up128(2 * chunk * g.period);
    // Packed edge batch: layer q's output differs from the stream's only in its first e_head[q] / last e_tail[q] rows (one more
    // per conv); its box holds those rows: tbox[q] = max(e_head, e_tail) (at least 4) rows, floor(128 / tbox) slots per MMA
    // tile.  The two rows next to them, which the next two layers read as well, are the stream's: the launch's store warps copy
    // them into the slot (with them inside the box, as before, the 256 / 512-channel stages ran 12 % more tiles) (rows of the box among them are replaced in the epilogue), so a slot is max(e_head, e_tail) + 2 rows.
    // (The last layer's interior rows are never read: no copies.)
    if (g.C % 128 == 0) {
      const int nl = (int)g.list.size();
      g.e_head.resize(nl); g.e_tail.resize(nl); g.tbox.assign(nl, 0);
      bool ok = true;
      int Pmax = 0;
      for (int q = 0; q < nl; ++q) {
        g.e_head[q] = hp / 2 + 1 + q;
        g.e_tail[q] = g.T - (Tp - tp) / 2 + q;
        // edge rows + the two copied rows; the stage's last layer is read at its edge rows only (next stage's gather, stitch, head)
        const int e_max = g.e_head[q] > g.e_tail[q] ? g.e_head[q] : g.e_tail[q];
        g.tbox[q] = e_max > 4 ? e_max : 4;          // (at most 32 = SH_SPARE_SLOTS boxes per tile)
        if (g.tbox[q] > 32 || e_max < 1 || 128 / g.tbox[q] > SH_SPARE_SLOTS) ok = false;   // (a half's last box overhangs by < 128 / tbox slots)
        const int slot_rows = q + 1 < nl ? (g.tbox[q] > e_max + 2 ? g.tbox[q] : e_max + 2) : g.tbox[q];
        if (slot_rows > Pmax) Pmax = slot_rows;
      }
      if (ok && g.T >= 2 * Pmax && g.e_head[nl - 1] == g.head && g.e_tail[nl - 1] == g.tail) {
        g.packed = true; g.P = Pmax;
        g.rows_edge = 2 * (chunk + SH_SPARE_SLOTS) * g.P;
      }
    }
    if (!g.packed && !shs.empty() && shs.back().packed) { pl.sh_head_on = false; break; }   // (a packed stage feeds packed stages only)
    shs.push_back(g);
    i0 = g.list.back() + 1; Tp = g.T; hp = g.head; tp = g.tail; shift_p = g.shift;
  }
  // A packed stage after a packed stage reads its input slots where the previous stage's last layer wrote them: that layer's
  // slots are made as long as the entry conv and the folded projection reach (P_in rows, an even number: the stride-2 view),
  // its store warps copy the stream rows past the edge rows, and the gather between the two stages is not launched.
  for (size_t g = 0; g < shs.size(); ++g) {
    SharedStage& h = shs[g];
    h.P_in = h.packed ? 2 * (h.tbox.size() > 1 ? h.tbox[1] : h.tbox[0] + 1) : 0;
    if (g == 0 || !h.packed || !shs[g - 1].packed) continue;
    SharedStage& a = shs[g - 1];
    int P2 = a.P > h.P_in ? a.P : h.P_in;
    P2 += P2 & 1;
    if (a.T < 2 * P2 || a.C != h.C_in) continue;
    a.P = P2; a.keep = h.P_in; a.rows_edge = 2 * (chunk + SH_SPARE_SLOTS) * a.P;
    h.in_place = true;
  }
  return pl;
}

aframe_status af_parse_layer_table(const void* host_blob, size_t bytes, int kernel_len, int n_channels,
                                   std::vector<LayerDesc>& layers, uint32_t hdr[8], const char** why);   // aframe_api.cu

// Host-only description of the plan above for a weight blob and a window spacing (include/aframe.h).
AF_API aframe_status aframe_describe_shared_plan(const void* host_blob, size_t bytes, int32_t kernel_len, int32_t n_channels,
                                                 int32_t window_spacing, int64_t n_windows, int32_t* first_stage_blocks,
                                                 aframe_stage_plan* stages, int32_t max_stages, int32_t* n_stages) {
  if (!host_blob || !first_stage_blocks || !n_stages || (max_stages > 0 && !stages) || kernel_len < 1 || window_spacing < 1 ||
      n_windows < 1 || max_stages < 0) return AFRAME_EINVAL;
  std::vector<LayerDesc> layers;
  uint32_t hdr[8];
  const char* why = "";
  const aframe_status st = af_parse_layer_table(host_blob, bytes, kernel_len, n_channels, layers, hdr, &why);
  if (st != AFRAME_OK) return st;
  *first_stage_blocks = 0; *n_stages = 0;
  if (layers.size() < 3 || layers[0].kind != 0 || layers[1].kind != 1) return AFRAME_OK;   // not a stem + pool table: nothing is shared
  const int64_t chunk = n_windows < tc_chunk_windows() ? n_windows : tc_chunk_windows();
  const SharedPlan pl = tc_plan_shared(layers, hdr[3] == 2, window_spacing, chunk);
  *first_stage_blocks = pl.s1_on ? pl.s1_k : 0;
  for (const SharedStage& g : pl.stages) {
    if (*n_stages >= max_stages) break;
    aframe_stage_plan& o = stages[(*n_stages)++];
    memset(&o, 0, sizeof(o));
    o.first_layer = g.i0; o.n_layers = (int32_t)g.list.size(); o.T = g.T; o.C = g.C; o.head = g.head; o.tail = g.tail;
    o.packed = g.packed ? 1 : 0; o.P = g.packed ? g.P : g.rows; o.spare_slots = g.packed ? SH_SPARE_SLOTS : 0;
    for (int q = 0; q < o.n_layers && q < 16; ++q) {
      o.e_head[q] = g.packed ? g.e_head[q] : 0; o.e_tail[q] = g.packed ? g.e_tail[q] : 0; o.tbox[q] = g.packed ? g.tbox[q] : 0;
    }
  }
  return AFRAME_OK;
}

aframe_status af_forward_bf16(aframe_ctx* ctx, const aframe_weights* w, const void* d_in, int in_dt, int64_t sB,
                              int64_t sT, const int64_t* choff, int64_t B, float* d_scores) {
  (void)sT;
  NetPlan plan;
  af_make_plan(w, true, plan);
  const int64_t chunk = tc_chunk_windows() < B ? tc_chunk_windows() : B;
  const size_t slot_bytes = ((plan.slot_elems * 2 * (size_t)chunk) + 1023) & ~(size_t)1023;
  const int n = (int)w->layers.size();
  SharedPlan shp = tc_plan_shared(w->layers, w->live_gn, sB, chunk);
  const int fuse = shp.fuse;
  const int n_part = fuse >= 0 ? (w->layers[fuse].t_out / 32) * (w->layers[fuse].c_out / 64) * TcCfg<256, true>::EPW : 0;   // head units of EPI_COLS channels
  // live GroupNorm scratch after the slots: (mu, rstd) per (window, group), then the conv epilogues' partial sums
  size_t gn_part_elems = 0;                                      // float2 per window
  if (w->live_gn)
    for (int i = 2; i < n; ++i) {
      const LayerDesc& l = w->layers[i];
      if (l.kind != 0) continue;
      const int u = l.c_out / w->n_groups < 32 ? l.c_out / w->n_groups : 32;   // (an upper bound on the units: 32-column units on the CTA-pair path)
      const size_t e = (size_t)(l.t_out / 32) * (l.c_out / u);
      if (e > gn_part_elems) gn_part_elems = e;
    }
  const size_t gn_stats_bytes = (sizeof(float2) * (size_t)w->n_groups * chunk + 1023) & ~(size_t)1023;
  const size_t part_bytes = w->live_gn ? gn_stats_bytes + ((sizeof(float2) * gn_part_elems * chunk + 1023) & ~(size_t)1023)
                                       : ((sizeof(float) * (size_t)n_part * chunk + 1023) & ~(size_t)1023);
  // shared first stage (see s1_gather_kernel): K streams + one gathered input + K edge results per chunk; shared later
  // stages (see sh_gather_kernel): per launched layer one stream and one edge-batch tensor, plus the gathered input
  const int s1_k = shp.s1_k;
  const bool s1_on = shp.s1_on;
  auto up128 = [](int64_t v) { return tc_up128(v); };
  std::vector<SharedStage>& shs = shp.stages;
  const bool sh_head_on = shp.sh_head_on;
  const bool s2_on = !shs.empty();
  const int64_t s1_rows = (chunk - 1) * (sB / 4) + w->layers[1].t_out;
  const size_t s1_stream_bytes = s1_on ? (((size_t)s1_rows * 128 + 1023) & ~(size_t)1023) : 0;
  const size_t s1_edge_bytes = s1_on ? (((size_t)2 * chunk * S1_PERIOD * 128 + 1023) & ~(size_t)1023) : 0;
  const size_t s1_bytes = (size_t)s1_k * s1_stream_bytes + (size_t)(s1_k + 1) * s1_edge_bytes;
  size_t s2_bytes = 0;
  for (size_t g = 0; g < shs.size(); ++g) {
    SharedStage& h = shs[g];
    // one tensor per layer: [stream rows | edge-batch rows], and the entry conv's input at twice the rows
    h.stream_bytes = ((size_t)(h.rows_stream + h.rows_edge) * h.C * 2 + 1023) & ~(size_t)1023;
    // the stage input: packed stages read the previous stage's stream in place and gather only the slots their first two
    // layers reach (P_in rows per slot at the previous stage's resolution); other stages gather [stream | short windows]
    h.x_bytes = h.in_place ? 0 : h.packed ? (((size_t)2 * (chunk + SH_SPARE_SLOTS) * h.P_in * h.C_in * 2 + 1023) & ~(size_t)1023)
                         : (((size_t)2 * (h.rows_stream + h.rows_edge) * h.C_in * 2 + 1023) & ~(size_t)1023);
    h.off = s2_bytes;
    s2_bytes += h.x_bytes + h.list.size() * h.stream_bytes;
  }
  aframe_status st = af_ws_reserve(ctx, ctx->ws_act, slot_bytes * plan.n_slots + part_bytes + s1_bytes + s2_bytes);
  if (st != AFRAME_OK) return st;
  char* base = reinterpret_cast<char*>(ctx->ws_act.ptr);
  char* s1_base = base + slot_bytes * plan.n_slots + part_bytes;
  auto s1_stream_ptr = [&](int k) { return reinterpret_cast<af_act_t*>(s1_base + (size_t)(k - 1) * s1_stream_bytes); };             // S_k, k = 1..K
  char* s2_base = s1_base + s1_bytes;
  auto sh_x_ptr = [&](int g) { return reinterpret_cast<af_act_t*>(s2_base + shs[g].off); };
  int64_t cur_nb = chunk;                          // windows of the chunk being planned / launched (row counts depend on it)
  auto sh_rows_stream = [&](int g) { return up128((cur_nb - 1) * shs[g].shift + shs[g].T); };
  auto sh_buf = [&](int g, int pass, int idx) {    // pass 0: the tensor (stream part first), 1: its edge-batch part; idx: position in the list
    const SharedStage& h = shs[g];
    return reinterpret_cast<af_act_t*>(s2_base + h.off + h.x_bytes + (size_t)idx * h.stream_bytes) + (pass ? sh_rows_stream(g) * h.C : 0);
  };
  auto s1_edge_ptr = [&](int k) { return reinterpret_cast<af_act_t*>(s1_base + (size_t)s1_k * s1_stream_bytes + (size_t)k * s1_edge_bytes); };  // X (k = 0), Y_k
  float* head_part = reinterpret_cast<float*>(base + slot_bytes * plan.n_slots);
  auto slot_ptr = [&](int layer) { return reinterpret_cast<af_act_t*>(base + slot_bytes * plan.slot[layer]); };
  if (!ctx->tc_cache) ctx->tc_cache = new std::vector<TcPlanCache>();
  std::vector<TcPlanCache>& caches = *static_cast<std::vector<TcPlanCache>*>(ctx->tc_cache);

  for (int64_t b0 = 0; b0 < B; b0 += chunk) {
    const int64_t nb = (B - b0 < chunk) ? (B - b0) : chunk;
    cur_nb = nb;
    TcPlanCache* pc = nullptr;
    for (auto& c : caches)
      if (c.w == w && c.base == base && c.nb == nb && c.slot_bytes == slot_bytes && c.win_stride == sB) { pc = &c; break; }
    if (!pc) {
      if (caches.size() > 8) caches.clear();
      caches.emplace_back();
      pc = &caches.back();
      pc->w = w; pc->base = base; pc->nb = nb; pc->slot_bytes = slot_bytes; pc->win_stride = sB;
      pc->launches.resize(n);
      pc->blocks.resize(n);
      pc->fused_with.assign(n, -1);
      pc->sc_of.assign(n, -1);
      pc->skip.assign(n, 0);
      // projection shortcut (1x1 conv, no ReLU, read only as layer i's residual): folded into layer i as extra K blocks,
      // which saves its launch, the write of its output and the residual read (the accumulation also stays in fp32)
      if (!w->live_gn)
        for (int i = 2; i < n; ++i) {
          const LayerDesc& l = w->layers[i];
          const int r = l.residual_from;
          if (l.kind != 0 || r < 2 || i == fuse || !has_projection_residual(w->layers, i) || !w->d_bias_sc[i]) continue;
          const LayerDesc& q = w->layers[r];
          bool ok = q.kind == 0 && q.k == 1 && q.pad == 0 && !q.relu && q.residual_from < 0 && q.c_in % 64 == 0 &&
                    q.t_out == l.t_out && q.c_out == l.c_out && q.t_in % q.stride == 0 && q.input_from >= 1 &&
                    l.k * (l.c_in / 64) + q.c_in / 64 <= 64;
          for (int j = 0; ok && j < n; ++j)
            if (j != i && (w->layers[j].input_from == r || w->layers[j].residual_from == r)) ok = false;
          if (w->layers[i].input_from == r) ok = false;
          if (ok) { pc->sc_of[i] = r; pc->skip[r] = 1; }
        }
      if (!w->live_gn)
        for (int i = 2; i < n; ++i) {
          const int ib = pc->fused_with[i] < 0 ? fusable_block(w, i) : -1;
          if (ib < 0) continue;
          // Shared stem: overlapping in-place windows (spacing a multiple of 4 samples, shorter than the window) whose
          // stem output is read only by this fused block: the stem runs ONCE over the whole stream, the block reads the
          // windows as strided views of it and patches the three rows per window that see the window's own zero padding.
          bool shared = i == 2 && w->layers[2].input_from == 1 && w->layers[ib].residual_from == 1 && nb >= 2 && sB % 4 == 0 &&
                        sB < w->layers[0].t_in;
          for (int j = 2; shared && j < n; ++j)
            if (j != 2 && j != ib && (w->layers[j].input_from == 1 || w->layers[j].residual_from == 1)) shared = false;
          const int64_t row_shift = shared ? sB / 4 : 0;
          const af_act_t* edge = slot_ptr(1) + ((nb - 1) * row_shift + w->layers[1].t_out) * 64;
          if (!build_block_launch(ctx, w, i, ib, slot_ptr(w->layers[i].input_from), slot_ptr(ib), nb, pc->blocks[ib], row_shift, edge)) { caches.pop_back(); return AFRAME_ECUDA; }
          if (shared) pc->shared_stem = true;
          pc->fused_with[i] = ib; pc->fused_with[ib] = i;
        }
      if (s1_on && pc->shared_stem && nb >= 2) {
        const int T1 = w->layers[1].t_out;
        const int64_t R0 = (nb - 1) * (sB / 4) + T1;
        pc->s1_stream.resize(s1_k + 1);
        pc->s1_edge.resize(s1_k + 1);
        bool ok = R0 < (1ll << 30) && 2 * nb * S1_PERIOD < (1ll << 30);
        for (int k = 1; ok && k <= s1_k; ++k) {
          const int ia = 2 * k, ib = 2 * k + 1;
          ok = build_block_launch(ctx, w, ia, ib, k == 1 ? slot_ptr(1) : s1_stream_ptr(k - 1), s1_stream_ptr(k), 1, pc->s1_stream[k], 0,
                                  nullptr, (int)R0) &&
               build_block_launch(ctx, w, ia, ib, s1_edge_ptr(0), s1_edge_ptr(k), 1, pc->s1_edge[k], 0, nullptr,
                                  (int)(2 * nb * S1_PERIOD), S1_PERIOD, S1_ROWS);
        }
        if (!ok) { caches.pop_back(); return AFRAME_ECUDA; }
        pc->s1_blocks = s1_k;
        pc->sh.resize(shs.size());
        for (size_t g = 0; ok && g < shs.size(); ++g) {
          const SharedStage& h = shs[g];
          TcPlanCache::SharedStagePlan& P = pc->sh[g];
          const int64_t rows_s = up128((nb - 1) * h.shift + h.T), rows_tot = rows_s + up128(2 * nb * h.period);
          auto idx_of = [&](int layer) { for (size_t q = 0; q < h.list.size(); ++q) if (h.list[q] == layer) return (int)q; return -1; };
          P.stream.resize(h.list.size());
          ok = rows_tot < (1ll << 30);
          P.packed = h.packed; P.P = h.P; P.nbp = nb + SH_SPARE_SLOTS;
          if (h.packed) { P.e_stride = h.P; P.e_tail0 = P.nbp * h.P; P.e_trow = h.T - h.P; }
          else { P.e_stride = 2 * h.period; P.e_tail0 = h.period; P.e_trow = h.T - h.rows; }
          if (h.packed) P.edge.resize(h.list.size());
          for (size_t q = 0; ok && h.packed && q < h.list.size(); ++q) {
            // packed edge batch: per layer one launch over the stream (one long window) and one over the short-window slots
            const int li = h.list[q];
            const LayerDesc& l = w->layers[li];
            const bool entry = li == h.i0;
            const int sc = pc->sc_of[li];
            const int qi = entry ? -1 : idx_of(l.input_from), qr = (l.residual_from >= 0 && sc < 0) ? idx_of(l.residual_from) : -1;
            ok = (entry || qi >= 0) && (l.residual_from < 0 || sc >= 0 || qr >= 0);
            if (!ok) break;
            // stage input: the previous stage's stream in place (its valid rows; the rest reads as zero), and the gathered slots
            const int q_prev = g ? (int)shs[g - 1].list.size() - 1 : 0;
            const af_act_t* x_stream = g ? sh_buf((int)g - 1, 0, q_prev) : s1_stream_ptr(s1_k);
            const af_act_t* x_edge = h.in_place ? sh_buf((int)g - 1, 1, q_prev) : sh_x_ptr((int)g);
            const int x_Pin = h.in_place ? shs[g - 1].P : h.P_in;
            TcShapeOverride ov_s{(int)rows_s, 0, 0, 0};
            TcShapeOverride ov_e{0, 0, 0, 0};
            const int64_t valid_prev = (g ? (nb - 1) * shs[g - 1].shift + shs[g - 1].T : (nb - 1) * (sB / 4) + w->layers[1].t_out) & ~(int64_t)1;
            if (entry) { ov_s.in_rows = valid_prev; ov_e.e_Pin = x_Pin; }
            if (sc >= 0) { ov_s.in_rows_sc = valid_prev; ov_e.e_Pin_sc = x_Pin; }
            // the conv that feeds the head stores nothing: its tensor holds the per-row head dot products instead
            // ([stream rows | edge-batch rows][C / 64] floats)
            const bool hr = sh_head_on && g + 1 == shs.size() && q + 1 == h.list.size();
            float* hr_s = reinterpret_cast<float*>(sh_buf((int)g, 0, (int)q));
            float* hr_e = hr_s + rows_s * (h.C / TcCfg<256, true>::EPI_COLS);
            ov_s.head_rows = ov_e.head_rows = hr;
            ov_s.pair_plan = ov_e.pair_plan = true;
            if (hr) pc->sh_head_rows = true;
            ov_e.e_nbp = (int)P.nbp; ov_e.e_P = h.P; ov_e.e_tbox = h.tbox[q]; ov_e.e_T = h.T; ov_e.e_head = h.e_head[q]; ov_e.e_tail = h.e_tail[q];
            ov_e.e_shift = h.shift; ov_e.e_nb = nb; const bool last_q = q + 1 == h.list.size();
            ov_e.e_stream = last_q && h.keep == 0 ? nullptr : sh_buf((int)g, 0, (int)q);
            ov_e.e_keep = last_q ? h.keep : 0;
            ok = build_launch(ctx, w, li, entry ? x_stream : sh_buf((int)g, 0, qi), qr >= 0 ? sh_buf((int)g, 0, qr) : nullptr,
                              sh_buf((int)g, 0, (int)q), 1, hr, hr_s, P.stream[q], sc, sc >= 0 ? x_stream : nullptr, &ov_s) &&
                 build_launch(ctx, w, li, entry ? x_edge : sh_buf((int)g, 1, qi), qr >= 0 ? sh_buf((int)g, 1, qr) : nullptr,
                              sh_buf((int)g, 1, (int)q), 1, hr, hr_e, P.edge[q], sc, sc >= 0 ? x_edge : nullptr, &ov_e);
          }
          for (size_t q = 0; ok && !h.packed && q < h.list.size(); ++q) {
            // one launch per layer over [stream | short windows]: the mask starts at the short windows (and their leading padding)
            const int li = h.list[q];
            const LayerDesc& l = w->layers[li];
            const TcShapeOverride ov{(int)rows_tot, h.period, h.rows, (int)rows_s};
            const bool entry = li == h.i0;
            const int sc = pc->sc_of[li];
            const af_act_t* in = entry ? sh_x_ptr((int)g) : sh_buf((int)g, 0, idx_of(l.input_from));
            const af_act_t* res = (l.residual_from >= 0 && sc < 0) ? sh_buf((int)g, 0, idx_of(l.residual_from)) : nullptr;
            ok = (entry || idx_of(l.input_from) >= 0) && (res == nullptr || idx_of(l.residual_from) >= 0) &&
                 build_launch(ctx, w, li, in, res, sh_buf((int)g, 0, (int)q), 1, false, nullptr, P.stream[q], sc,
                              sc >= 0 ? sh_x_ptr((int)g) : nullptr, &ov);
          }
          P.layers = h.list;
          P.T = h.T; P.C = h.C; P.C_in = h.C_in; P.head = h.head; P.tail = h.tail; P.shift = h.shift; P.rows = h.rows; P.period = h.period;
        }
        if (!ok) { caches.pop_back(); return AFRAME_ECUDA; }
        pc->sh_head = sh_head_on;
      }
      for (int i = 2; i < n; ++i) {
        const LayerDesc& l = w->layers[i];
        if (l.kind != 0 || pc->fused_with[i] >= 0 || pc->skip[i]) continue;
        const int sc = pc->sc_of[i];
        if (!build_launch(ctx, w, i, slot_ptr(l.input_from),
                          l.residual_from >= 0 && !w->live_gn && sc < 0 ? slot_ptr(l.residual_from) : nullptr, slot_ptr(i), nb,
                          i == fuse, head_part, pc->launches[i], sc, sc >= 0 ? slot_ptr(w->layers[sc].input_from) : nullptr)) {
          caches.pop_back(); return AFRAME_ECUDA;
        }
        if (w->live_gn) {
          // statistics from the epilogue's fp32 accumulators when a warp's 32 rows are one slab of one window and a group
          // is a whole number of 8..64-column units; else af_launch_gn_bf16 reads z back
          const int cg = l.c_out / w->n_groups;
          const int ec = pc->launches[i].cg2 ? TcCfg<256, true>::EPI_COLS : 64;   // accumulator columns per epilogue thread
          const int u = cg < ec ? cg : ec;
          TcConvParams& pp = pc->launches[i].p;
          if (pp.T_box % 32 == 0 && (u == 8 || u == 16 || u == 32 || u == 64) && cg % u == 0) {
            pp.gn_part = reinterpret_cast<float2*>(reinterpret_cast<char*>(head_part) + gn_stats_bytes);
            pp.gn_unit = u;
          }
        }
      }
    }
    const size_t esz = af_dt_bytes(in_dt);
    std::vector<cudaEvent_t> lev;
    if (ctx->layer_ms) {
      lev.resize(n + 1);
      for (auto& e : lev) cudaEventCreate(&e);
      cudaEventRecord(lev[0], ctx->stream);
    }
    af_prof_begin(ctx, AFRAME_PROF_STEM);
    // (a tcgen05 formulation of the stem -- three K = 16 MMAs on an im2col tile, pool = max of three accumulators -- was
    //  built and measured: no faster end to end than this fp32 CUDA-core kernel under the power cap, and less accurate
    //  because its operands are bf16; it was dropped)
    float2* gn_stats = reinterpret_cast<float2*>(head_part);     // live GroupNorm: the scratch after the slots holds (mu, rstd)
    const StemGn sgn{gn_stats, w->d_gamma[0], w->d_beta[0], w->n_groups, w->gn_eps};
    if (pc->shared_stem)
      st = af_launch_stem_stream_bf16(ctx, w->layers[0], w->layers[1], reinterpret_cast<const char*>(d_in) + (size_t)(b0 * sB) * esz,
                                      in_dt, sB, choff, w->d_w32[0], w->d_bias[0], nb, slot_ptr(1),
                                      slot_ptr(1) + ((nb - 1) * (sB / 4) + w->layers[1].t_out) * 64);
    else
    st = af_launch_stem_bf16(ctx, w->layers[0], w->layers[1], reinterpret_cast<const char*>(d_in) + (size_t)(b0 * sB) * esz,
                             in_dt, sB, choff, w->d_w32[0], w->d_bias[0], nb, slot_ptr(1), w->live_gn ? &sgn : nullptr);
    af_prof_end(ctx, AFRAME_PROF_STEM, 1);
    if (st != AFRAME_OK) return st;
    int n_conv = 0, span_conv = 0;             // conv launches so far (tile direction) / in the open timing span
    // gathers, stitches and the head-rows sum are timed apart from the convolutions (AFRAME_PROF_GATHER)
    auto aux_begin = [&]() { af_prof_end(ctx, AFRAME_PROF_CONV, span_conv); span_conv = 0; af_prof_begin(ctx, AFRAME_PROF_GATHER); };
    auto aux_end = [&]() { af_prof_end(ctx, AFRAME_PROF_GATHER, 1); af_prof_begin(ctx, AFRAME_PROF_CONV); };
    if (ctx->layer_ms) { cudaEventRecord(lev[1], ctx->stream); cudaEventRecord(lev[2], ctx->stream); }
    if (pc->s1_blocks > 0) {
      // shared first stage: per block one pass over the stream and one over the short edge windows, then the stitch
      af_prof_begin(ctx, AFRAME_PROF_CONV);
      const int T1 = w->layers[1].t_out, K = pc->s1_blocks;
      const int64_t shift = sB / 4;
      const uint4* E0 = reinterpret_cast<const uint4*>(slot_ptr(1) + ((nb - 1) * shift + T1) * 64);
      for (int k = 1; k <= K; ++k) {
        cudaError_t e = launch_block(pc->s1_stream[k], ctx->stream);
        ctx->launches++; ++n_conv; ++span_conv; ctx->tc_macs += pc->s1_stream[k].macs;
        if (e != cudaSuccess) { snprintf(ctx->err, sizeof(ctx->err), "conv_block (stream) launch: %s", cudaGetErrorString(e)); return AFRAME_ECUDA; }
        const int64_t n_g = 2 * nb * S1_PERIOD * 8;
        aux_begin();
        s1_gather_kernel<<<(unsigned)((n_g + 255) / 256), 256, 0, ctx->stream>>>(
            reinterpret_cast<uint4*>(s1_edge_ptr(0)), reinterpret_cast<const uint4*>(k == 1 ? slot_ptr(1) : s1_stream_ptr(k - 1)),
            k == 1 ? nullptr : reinterpret_cast<const uint4*>(s1_edge_ptr(k - 1)), k == 1 ? E0 : nullptr, nb, T1, shift, 2 * k, 2 * k - 1);
        AF_LAUNCH_CHECK(ctx);
        aux_end();
        e = launch_block(pc->s1_edge[k], ctx->stream);
        ctx->launches++; ++n_conv; ++span_conv; ctx->tc_macs += pc->s1_edge[k].macs;
        if (e != cudaSuccess) { snprintf(ctx->err, sizeof(ctx->err), "conv_block (edge) launch: %s", cudaGetErrorString(e)); return AFRAME_ECUDA; }
      }
      if (pc->sh.empty()) {
        const int64_t n_s = nb * T1 * 8;
        aux_begin();
        s1_stitch_kernel<<<(unsigned)((n_s + 255) / 256), 256, 0, ctx->stream>>>(
            reinterpret_cast<uint4*>(slot_ptr(2 * K + 1)), reinterpret_cast<const uint4*>(s1_stream_ptr(K)),
            reinterpret_cast<const uint4*>(s1_edge_ptr(K)), nb, T1, shift, 2 * K + 2, 2 * K + 1);
        AF_LAUNCH_CHECK(ctx);
        aux_end();
      }
      // shared later stages: each reads the previous stage's stream and edge results directly; only the last one is stitched
      for (size_t g = 0; g < pc->sh.size(); ++g) {
        TcPlanCache::SharedStagePlan& P = pc->sh[g];
        const int64_t n_short = 2 * nb, edge_rows_in = 2 * up128(2 * nb * P.period);
        const int pieces_in = P.C_in / 8;
        const int64_t copy_rows = 2 * sh_rows_stream((int)g);
        const int64_t n_g = (copy_rows + edge_rows_in) * pieces_in;
        const int q_prev = g ? (int)pc->sh[g - 1].layers.size() - 1 : 0;
        if (P.packed) {
          const int P_in = shs[g].P_in;
          const int64_t n_p = (2 * P.nbp * P_in) * pieces_in;
          if (!shs[g].in_place) {
          aux_begin();
          shp_gather_kernel<<<(unsigned)((n_p + 255) / 256), 256, 0, ctx->stream>>>(
              reinterpret_cast<uint4*>(sh_x_ptr((int)g)),
              reinterpret_cast<const uint4*>(g ? sh_buf((int)g - 1, 0, q_prev) : s1_stream_ptr(K)),
              reinterpret_cast<const uint4*>(g ? sh_buf((int)g - 1, 1, q_prev) : s1_edge_ptr(K)), nb, P.nbp, 2 * P.T, pieces_in,
              2 * P.shift, g ? pc->sh[g - 1].e_stride : 2 * S1_PERIOD, g ? pc->sh[g - 1].e_tail0 : S1_PERIOD,
              g ? pc->sh[g - 1].e_trow : T1 - S1_ROWS, g ? pc->sh[g - 1].head : 2 * K + 2, g ? pc->sh[g - 1].tail : 2 * K + 1,
              0, 0, P_in);
          AF_LAUNCH_CHECK(ctx);
          aux_end();
          }
          // Launch order: stream(0) | edge(q) with stream(q + 1) as ONE launch of two problems (independent of each other: both
          // need stream(q), and edge(q) needs edge(q - 1)) | ... | edge(last).  A stream launch alone costs 16-30 us for 1/8 of an
          // edge launch's work (profiles/r01i_conv_full.md); as the second problem its tiles fill the edge launch's last wave.
          const size_t nl = P.layers.size();
          auto can_pair = [&](size_t q) {
            if (q + 1 >= nl) return false;
            const TcLaunch& a = P.edge[q];
            const TcLaunch& b = P.stream[q + 1];
            return a.cg2 && b.cg2 && a.BN == 256 && b.BN == 256 && !a.head && !b.head && !a.halo && !b.halo && a.p.stages == b.p.stages &&
                   a.p.nbuf == b.p.nbuf && a.p.pf == b.p.pf && a.smem == b.smem && a.p.c_out == b.p.c_out;
          };
          // consecutive edge launches walk their tiles in opposite directions: layer q + 1 starts on the slots layer q wrote
          // last, which are still in L2 (an edge-batch tensor is 100-135 MB, the L2 126 MB)
          auto launch_one = [&](TcLaunch& A, TcLaunch* B2, int rev = 0) -> aframe_status {
            A.p.reverse = rev;
            if (B2) B2->p.reverse = 0;
            cudaError_t e = launch_conv(A, ctx->stream, B2);
            ctx->launches++; ++n_conv; ++span_conv; ctx->tc_macs += A.macs + (B2 ? B2->macs : 0.0);
            if (e != cudaSuccess) { snprintf(ctx->err, sizeof(ctx->err), "conv_tc (packed edge stage) launch: %s", cudaGetErrorString(e)); return AFRAME_ECUDA; }
            return AFRAME_OK;
          };
          if ((st = launch_one(P.stream[0], nullptr)) != AFRAME_OK) return st;
          for (size_t q = 0; q < nl; ++q) {
            if (can_pair(q)) {
              if ((st = launch_one(P.edge[q], &P.stream[q + 1], (int)(q & 1))) != AFRAME_OK) return st;
            } else {
              if ((st = launch_one(P.edge[q], nullptr, (int)(q & 1))) != AFRAME_OK) return st;
              if (q + 1 < nl && (st = launch_one(P.stream[q + 1], nullptr)) != AFRAME_OK) return st;
            }
          }
        } else {
        aux_begin();
        sh_gather_kernel<<<(unsigned)((n_g + 255) / 256), 256, 0, ctx->stream>>>(
            reinterpret_cast<uint4*>(sh_x_ptr((int)g)),
            reinterpret_cast<const uint4*>(g ? sh_buf((int)g - 1, 0, q_prev) : s1_stream_ptr(K)),
            reinterpret_cast<const uint4*>(g ? sh_buf((int)g - 1, 1, q_prev) : s1_edge_ptr(K)), nb, n_short, 2 * P.T, pieces_in,
            2 * P.shift, g ? pc->sh[g - 1].period : S1_PERIOD, g ? pc->sh[g - 1].rows : S1_ROWS, g ? pc->sh[g - 1].head : 2 * K + 2,
            g ? pc->sh[g - 1].tail : 2 * K + 1, copy_rows, g ? sh_rows_stream((int)g - 1) : (nb - 1) * shift + T1, P.rows, P.period,
            edge_rows_in);
        AF_LAUNCH_CHECK(ctx);
        aux_end();
        for (size_t q = 0; q < P.layers.size(); ++q) {
          TcLaunch& L2 = P.stream[q];
          L2.p.reverse = 0;
          cudaError_t e = launch_conv(L2, ctx->stream);
          ctx->launches++; ++n_conv; ++span_conv; ctx->tc_macs += L2.macs;
          if (e != cudaSuccess) { snprintf(ctx->err, sizeof(ctx->err), "conv_tc (shared stage) launch: %s", cudaGetErrorString(e)); return AFRAME_ECUDA; }
        }
        }
        if (g + 1 == pc->sh.size() && pc->sh_head && pc->sh_head_rows) {
          const int q_last = (int)P.layers.size() - 1;
          const int hu = P.C / TcCfg<256, true>::EPI_COLS;          // head units per row
          const int64_t n_warps = nb * (P.T / 32);
          const float* hr_s = reinterpret_cast<const float*>(sh_buf((int)g, 0, q_last));
          aux_begin();
          sh_head_rows_kernel<<<(unsigned)((n_warps + 7) / 8), 256, 0, ctx->stream>>>(
              hr_s, sh_rows_stream((int)g), hr_s + sh_rows_stream((int)g) * hu, 2 * P.nbp * P.P, head_part, nb, P.T, hu, P.shift,
              P.head, P.tail, P.e_stride, P.e_tail0, P.e_trow);
          AF_LAUNCH_CHECK(ctx);
          aux_end();
        } else if (g + 1 == pc->sh.size()) {
          const int last = P.layers.back(), q_last = (int)P.layers.size() - 1, pieces = P.C / 8;
          const int64_t n_s = nb * P.T * pieces;
          aux_begin();
          s2_stitch_kernel<<<(unsigned)((n_s + 255) / 256), 256, 0, ctx->stream>>>(
              reinterpret_cast<uint4*>(slot_ptr(last)), reinterpret_cast<const uint4*>(sh_buf((int)g, 0, q_last)),
              reinterpret_cast<const uint4*>(sh_buf((int)g, 1, q_last)), nb, P.T, pieces, P.shift, P.head, P.tail, P.e_stride, P.e_tail0, P.e_trow);
          AF_LAUNCH_CHECK(ctx);
          aux_end();
        }
      }
    }
    for (int i = 2; i < n; ++i) {
      const LayerDesc& l = w->layers[i];
      struct Rec { aframe_ctx* c; std::vector<cudaEvent_t>& v; int i; ~Rec() { if (c->layer_ms) cudaEventRecord(v[i + 1], c->stream); } } rec{ctx, lev, i};
      if (i < 2 + 2 * pc->s1_blocks) continue;                 // ran in shared form above
      if (!pc->sh.empty() && i <= pc->sh.back().layers.back()) continue;
      if (l.kind == 0 && pc->fused_with[i] > i) continue;      // first conv of a fused block: runs with its partner
      if (pc->skip[i]) continue;                               // projection shortcut: runs inside the conv it feeds
      if (l.kind == 0) {
        // Alternate the direction in which consecutive launches walk their tiles: a layer then starts with the rows its
        // producer wrote LAST, which are still in L2 (walking every layer forwards evicts exactly the lines that are
        // about to be read).
        const int rev = n_conv & 1;
        pc->launches[i].p.reverse = rev;
        pc->blocks[i].p.reverse = rev;
        const TcLaunch& L = pc->launches[i];
        af_prof_begin(ctx, AFRAME_PROF_CONV);
        ++n_conv; ++span_conv;
        cudaError_t e = pc->fused_with[i] >= 0 ? launch_block(pc->blocks[i], ctx->stream) : launch_conv(L, ctx->stream);
        ctx->launches++; ctx->tc_macs += pc->fused_with[i] >= 0 ? pc->blocks[i].macs : L.macs;
        if (e != cudaSuccess) { snprintf(ctx->err, sizeof(ctx->err), "conv_tc launch: %s", cudaGetErrorString(e)); return AFRAME_ECUDA; }
        if (w->live_gn) {
          st = af_launch_gn_bf16(ctx, slot_ptr(i), l.residual_from >= 0 ? slot_ptr(l.residual_from) : nullptr, l.t_out, l.c_out,
                                 w->n_groups, w->gn_eps, w->d_gamma[i], w->d_beta[i], l.relu, nb, gn_stats, L.p.gn_part, L.p.gn_unit);
          if (st != AFRAME_OK) return st;
        }
      } else if (l.kind == 2) {
        af_prof_end(ctx, AFRAME_PROF_CONV, span_conv);
        n_conv = 0; span_conv = 0;
        af_prof_begin(ctx, AFRAME_PROF_HEAD);
        if (fuse >= 0) {
          head_finish_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, ctx->stream>>>(head_part, n_part, 1.0f / l.t_in, w->head_b, nb,
                                                                                  d_scores + b0);
          ctx->launches++;
          if (cudaGetLastError() != cudaSuccess) return af_fail(ctx, AFRAME_ECUDA, "head_finish launch failed");
        } else {
          st = af_launch_head(ctx, slot_ptr(l.input_from), AF_DT_F16, w->d_head_w, w->head_b, l.t_in, l.c_in, nb, d_scores + b0);
        }
        af_prof_end(ctx, AFRAME_PROF_HEAD, 1);
        if (st != AFRAME_OK) return st;
      }
    }
    if (ctx->layer_ms) {
      cudaStreamSynchronize(ctx->stream);
      for (int i = 0; i < n; ++i) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, lev[i], lev[i + 1]);
        ctx->layer_ms[i] += ms;
      }
      for (auto& e : lev) cudaEventDestroy(e);
    }
  }
  return AFRAME_OK;
}
