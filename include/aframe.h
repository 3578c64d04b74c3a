/* aframe.h -- C ABI of the B200-native (sm_100a) Aframe streaming detection statistic.
 *
 * Method: arXiv 2403.18661 (Marx et al. 2024), cited below as P:<line of PAPER.md>.
 *   strain [2][N] @ 2048 Hz  ->  Welch PSD  ->  whitening filter  ->  whitened stream
 *   ->  overlapping windows  ->  1D ResNet  ->  one scalar per window
 * (Sec. II network; Sec. IV.B "PSD estimation, filter construction, and whitening";
 *  P:170-172 Sec. VI snapshotter -> whitener -> network; Sec. IX timeslides.)
 * The parameters the paper leaves open are the readings A1..C3 of DESIGN.md.
 *
 * Conventions
 *  - Pointers named d_* are DEVICE pointers owned by the caller; the library never frees or
 *    reallocates them.  Pointers named h_* / `host_*` are HOST pointers.
 *  - All work is enqueued on the CUDA stream given to aframe_create.  No call synchronises the
 *    stream except aframe_create / aframe_destroy / aframe_weights_load / *_create / *_destroy
 *    and a call that has to grow the context's internal workspace (first use at a larger size).
 *  - Every call returns an aframe_status; none throws, aborts or prints.  aframe_last_error
 *    returns a context-owned, NUL-terminated description of the last failure.
 *  - No CPU fallback exists: on a device that is not compute capability 10.x aframe_create
 *    returns AFRAME_EUNSUPPORTED.
 *  - Threads: a context and the weights / stream objects created from it may be used by one host
 *    thread at a time; different contexts share no mutable state and may be used concurrently.
 *  - NaN/Inf in the inputs propagate to the outputs; they are not trapped.
 *  - Strain is pre-scaled on load by the exact power of two 2^strain_scale_log2 (reading A9:
 *    a PSD of ~1e-46 is below the smallest fp32 denormal).  PSDs handed out by the library are
 *    in SCALED units: true PSD * 2^(2*strain_scale_log2).  Whitened output is unit-free and
 *    unaffected.
 */
#ifndef AFRAME_H_
#define AFRAME_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  AFRAME_OK = 0,
  AFRAME_EINVAL = 1,       /* bad parameter value (NULL pointer, non power-of-two FFT length, ...) */
  AFRAME_ESHAPE = 2,       /* sizes inconsistent with the configuration / layer table          */
  AFRAME_ENOMEM = 3,       /* host or device allocation failed                                  */
  AFRAME_ECUDA = 4,        /* a CUDA call failed; aframe_last_error holds the CUDA string       */
  AFRAME_ESTATE = 5,       /* object used in a state that does not allow the call               */
  AFRAME_EUNSUPPORTED = 6  /* device is not sm_100, or the layer table needs an unsupported op  */
} aframe_status;

/* Two uses.
 * (1) cfg.precision, the arithmetic of the network path: AFRAME_FP32 (CUDA-core FFMA) or AFRAME_F16, the tensor-core
 *     path (tcgen05 kind::f16): folded weights rounded once to IEEE half, every stored activation rounded once to half
 *     (round to nearest even, saturating at +-65504; NaN stays NaN), products exact, accumulation, bias, residual add and
 *     ReLU in fp32, stem arithmetic and head in fp32 (reading B10 of DESIGN.md).  AFRAME_BF16 is refused here
 *     (AFRAME_EUNSUPPORTED): with bf16 storage the scores lose their rank order -- Spearman 0.9987 against the float64
 *     oracle on BASELINE.json configs[1], measured, which IS the ceiling of that format (0.9985 for the oracle with
 *     bf16 roundings) and below the 0.999 the contract asks for -- while half costs the same bytes and the same
 *     tensor-core rate and gives > 0.9999.
 * (2) the element type of a whitened stream handed in or out (out_dtype / dtype arguments): any of the three. */
typedef enum { AFRAME_FP32 = 0, AFRAME_BF16 = 1, AFRAME_F16 = 2 } aframe_precision;

/* POD configuration, versioned by .size (= sizeof(aframe_config)).  Defaults in comments are
 * BASELINE.json configs[1..4]; configs[0] uses n_design 4096, kernel_len 2048. */
typedef struct {
  uint32_t size;
  int32_t  n_channels;        /* 2: channel 0 = H1, 1 = L1                         */
  double   fs;                /* 2048 Hz                                                  */
  int32_t  welch_nfft;        /* 4096 = 2 s Welch segment (reading A1); power of two, 1024..8192 */
  int32_t  welch_hop;         /* 2048 = 50 % overlap; must equal welch_nfft/2                    */
  int32_t  filter_len;        /* L = 2048 = 1 s: 0.5 s corrupted per edge; <= 4096*/
  int32_t  n_design;          /* N_d design-grid FFT length (reading A4): power of two, <= 8192  */
  double   f_lo, f_hi;        /* 20, 1000 Hz inclusive band (reading A3)                         */
  int32_t  kernel_len;        /* K = 3072 = 1.5 s window                                 */
  int32_t  stride;            /* s = 128 samples = 16 Hz inference rate (paper: 512 = 4 Hz)*/
  int64_t  psd_len;           /* 131072 = 64 s of PSD history; multiple of welch_hop     */
  int64_t  psd_update;        /* 16384 = new PSD every 8 s (BASELINE.json configs[2])            */
  int32_t  strain_scale_log2; /* 70                                                              */
  int32_t  precision;         /* network path: AFRAME_F16 (tensor cores, default) or AFRAME_FP32 */
  int32_t  welch_average;     /* 0 = mean over segments (reading A1, default); 1 = per-bin median
                                 divided by its bias for n segments (NEXT-3 variant; n <= 255)   */
  int32_t  stream_full_forward; /* aframe_stream_step: 0 (default) = the incremental network where the configuration
                                 allows it (see aframe_stream_incremental), on a cluster of 16 CTAs if the device can place
                                 one, else 8; 1 = one full forward of the window per update; 2 = the incremental network on
                                 the portable cluster size 8 */
} aframe_config;

typedef struct aframe_ctx aframe_ctx;
typedef struct aframe_weights aframe_weights;
typedef struct aframe_stream_state aframe_stream_state;

/* Fill *cfg with the defaults above (size set).  Never fails for cfg != NULL. */
aframe_status aframe_config_default(aframe_config* cfg);

/* Create a context bound to the current CUDA device and to `cuda_stream` (a cudaStream_t; NULL = the
 * legacy default stream).  Validates cfg on the host (AFRAME_EINVAL / AFRAME_ESHAPE), checks the
 * device (AFRAME_EUNSUPPORTED) and uploads twiddle/window tables.  Synchronises. */
aframe_status aframe_create(const aframe_config* cfg, void* cuda_stream, aframe_ctx** out);
void          aframe_destroy(aframe_ctx* ctx);
const char*   aframe_last_error(const aframe_ctx* ctx);   /* ctx may be NULL: returns a static string */

/* ---- O-1  Welch PSD ("The first 8 s is used to estimate the PSD"; reading A1) -------
 * d_strain: [C][ld] fp32 raw strain, channel c at d_strain + c*ld, n_samples valid per channel
 *           (n_samples >= welch_nfft, else AFRAME_ESHAPE).
 * d_psd   : [C][welch_nfft/2+1] fp32, one-sided density, SCALED units, mean over the
 *           floor((n_samples-nfft)/hop)+1 Hann-windowed, mean-detrended segments (cfg.welch_average
 *           = 1: their per-bin median over its bias; at most 255 segments, else AFRAME_EUNSUPPORTED). */
aframe_status aframe_psd_welch(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                               float* d_psd);

/* The same PSD (same kernels, bit-identical result) for callers that may not allocate device memory -- code under CUDA-graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc: the periodogram scratch is a file-scope device array of
 * aframe_psd_welch_static_max_floats() = 2 * 64 * 2049 floats (1.0 MiB, held by every GPU that loads the library until
 * the process exits), so the call performs no cudaMalloc / cudaFree and calls no allocating routine.
 * AFRAME_ESHAPE (with the sizes in aframe_last_error) if n_channels * segments * (welch_nfft / 2 + 1) exceeds that;
 * AFRAME_ESTATE if the context's device is not the current device.  Arguments as aframe_psd_welch.
 * The array is shared by every call, context and stream on the device and keeps the last call's contents (nothing in it has
 * to start at zero: a call writes every periodogram before it reads it); calls that overlap on the GPU race on it, so
 * serialise them (one stream, or events between streams). */
aframe_status aframe_psd_welch_static(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                      float* d_psd);
int64_t       aframe_psd_welch_static_max_floats(void);

/* ---- O-2/O-3  filter design + whitening (readings A3-A6) -----------------------------
 * Designs the L-tap zero-phase FIR whitening filter from d_psd (as returned by aframe_psd_welch) and
 * applies it to a contiguous segment by FFT overlap-save.  Output has n_samples - filter_len samples
 * per channel: out[c][m] corresponds to input sample m + filter_len/2 (0.5 s cropped per edge).
 * d_out: [C][ld_out] of fp32, bf16 or fp16 (out_dtype).  n_samples <= filter_len writes nothing (OK). */
aframe_status aframe_whiten(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                            const float* d_psd, void* d_out, int64_t ld_out, aframe_precision out_dtype);

/* ---- the batched real transform of the overlap-save block, on its own ------------------------------------------------
 * BASELINE.json's north_star names "a batched power-of-two real FFT/iFFT" as a subsystem; inside aframe_whiten it is fused
 * with the spectral multiply ("whitened in the frequency-domain, and transformed back to time-domain").  These two
 * calls run exactly its two halves, one row per 8192-sample block, so the transform can be tested and profiled alone.
 * d_x   : [batch][8192] fp32 real rows, contiguous, 8-byte aligned.
 * d_spec: [batch][4097][2] fp32 (re, im), the one-sided spectrum X[k] = sum_n x[n] exp(-2 pi i n k / 8192), k = 0..4096.
 * aframe_irfft8192 carries the 1/8192 (x = irfft(rfft(x))) and ignores Im X[0] and Im X[4096].  batch = 0 is a no-op. */
aframe_status aframe_rfft8192(aframe_ctx* ctx, const float* d_x, int64_t batch, float* d_spec);
aframe_status aframe_irfft8192(aframe_ctx* ctx, const float* d_spec, int64_t batch, float* d_x);

/* Optional read-back of the taps designed by the last aframe_whiten call on this context:
 * d_taps [C][filter_len+1] fp32, h[j + L/2], j = -L/2..L/2 (used by the parity tests of O-2). */
aframe_status aframe_filter_taps(aframe_ctx* ctx, float* d_taps);

/* ---- O-6  rolling-PSD whitening of a long segment (BASELINE.json configs[2], [3]) -----------------
 * Same result, sample for sample, as feeding the segment through aframe_stream_step: a new PSD every
 * psd_update samples from the trailing psd_len samples, each whitened sample m using the filter of
 * epoch floor((stride*(floor((m+L/2)/stride)+1) - psd_len)/psd_update).  The first output corresponds
 * to raw sample psd_len - stride - L/2; *h_n_out (HOST pointer) receives the samples written per
 * channel (0 if n_samples < psd_len).  d_out: [C][ld_out]. */
aframe_status aframe_whiten_rolling(aframe_ctx* ctx, const float* d_strain, int64_t n_samples, int64_t ld,
                                    void* d_out, int64_t ld_out, aframe_precision out_dtype,
                                    int64_t* h_n_out);

/* ---- NEXT-4  training-time whitening batch -------------------------------------------------
 * "The length of each noise window sampled from disk is 10.5 s.  The first 8 s is used to estimate the
 * power spectral density (PSD) used for whitening.  The remaining 2.5 s of the window is whitened [...]
 * 0.5 s of data is corrupted on both ends of the window and removed."  Every (element, detector) row gets
 * its OWN Welch PSD (from its first n_psd samples), its own filter (O-2) and is whitened (O-3) over its
 * remaining n_samples - n_psd samples.
 * d_strain: [n_batch][C][n_samples] fp32, contiguous.  d_out: [n_batch][C][n_samples - n_psd - filter_len]
 * fp32, bf16 or fp16, contiguous (the paper's shapes: n_samples 21504, n_psd 16384 -> 3072 = kernel_len).
 * AFRAME_ESHAPE if n_psd < welch_nfft, n_samples - n_psd <= filter_len or n_batch * C > 65535. */
aframe_status aframe_whiten_batch(aframe_ctx* ctx, const float* d_strain, int64_t n_batch, int64_t n_samples,
                                  int64_t n_psd, void* d_out, aframe_precision out_dtype);

/* ---- NEXT-4  false-alarm rate of events against a background ------------------------
 * "a false alarm rate (FAR) can be assigned to injected events by dividing the number of background
 * events with detection statistic greater than the event of interest, with livetime analyzed."
 * d_background: [n_bg] fp32 detection statistics of the background triggers (timeslides), any order.
 * d_events    : [n_ev] fp32.   d_counts: [n_ev] int64, number of background values STRICTLY greater
 * (NaN compares false).  d_far: [n_ev] fp64 = counts / livetime_s in 1/s, or NULL.  n_bg = 0 gives
 * zeros; n_ev = 0 is a no-op.  AFRAME_EINVAL if livetime_s <= 0 while d_far != NULL. */
aframe_status aframe_far(aframe_ctx* ctx, const float* d_background, int64_t n_bg, const float* d_events,
                         int64_t n_ev, double livetime_s, int64_t* d_counts, double* d_far);

/* ---- weights (readings B1-B7) ----------------------------------------------------------
 * host_blob: the version-1 blob documented in synthdata/weights.py (header, layer table, UNFOLDED
 * fp32 parameters).  The library validates the table against cfg (AFRAME_ESHAPE), folds the frozen
 * norm into (W', b') in double precision, and uploads fp32 and fp16 (K-major) copies.  Synchronises.
 * Blob norm_kind 2 (NEXT-2, P:39 true GroupNorm) carries no frozen statistics: nothing is folded, and
 * aframe_forward computes mean / variance per window and group on the device after every conv. */
aframe_status aframe_weights_load(aframe_ctx* ctx, const void* host_blob, size_t bytes, aframe_weights** out);
void          aframe_weights_free(aframe_weights* w);

/* ---- O-5  network forward ------------------------------------------------------------------------------
 * d_windows: [B][C][kernel_len] fp32, already whitened.  d_scores: [B] fp32 raw logits (no sigmoid, B8).
 * B <= 0 is AFRAME_EINVAL.  Precision follows cfg.precision (AFRAME_F16: tcgen05 tensor-core path, fp16 weights and
 * activations, fp32 accumulation, reading B10; AFRAME_FP32: CUDA-core FFMA path). */
aframe_status aframe_forward(aframe_ctx* ctx, const aframe_weights* w, const float* d_windows, int64_t B,
                             float* d_scores);

/* Same network, windows taken in place from a whitened stream (O-4, no unfold copy; timeslides C3):
 * window i, channel c = d_white[c*ld + first + i*stride + chan_shift[c] + (0..kernel_len)).
 * dtype is the element type of d_white; chan_shift is a HOST array of n_channels entries (NULL = 0). */
aframe_status aframe_forward_strided(aframe_ctx* ctx, const aframe_weights* w, const void* d_white,
                                     aframe_precision dtype, int64_t ld, int64_t first,
                                     const int64_t* chan_shift, int64_t B, float* d_scores);

/* ---- O-6  streaming ("snapshotting") -------------------------------------------------
 * The state (raw ring, cached periodograms, PSD, filter, whitened ring, activations) is an opaque
 * device-resident object owned by the library.  aframe_stream_create returns AFRAME_ESHAPE unless cfg.stride divides
 * cfg.welch_hop (one Welch segment completes exactly on an update) and psd_len >= stride + filter_len.
 * Lifetime: the natural order is states, weights, context.  Other orders are safe: aframe_destroy releases the device
 * resources of the weights and stream states that are still alive and leaves them as dead shells, and aframe_weights_free
 * does the same to the stream states built on those weights; a dead shell only accepts its own free / destroy call
 * (aframe_stream_step on one returns AFRAME_ESTATE, a forward with dead weights AFRAME_ESTATE).
 * aframe_stream_step replays one captured CUDA graph per (d_new_samples, d_scores, d_n_scores) triple and keeps the four
 * most recently used: a caller should cycle through at most four sets of buffers. */
aframe_status aframe_stream_create(aframe_ctx* ctx, const aframe_weights* w, aframe_stream_state** out);
aframe_status aframe_stream_reset(aframe_stream_state* st);
void          aframe_stream_destroy(aframe_stream_state* st);

/* One update: d_new_samples [C][stride] fp32 raw strain.  Writes d_n_scores[0] (0 during warm-up,
 * else 1) and, when 1, d_scores[0].  CUDA-graph capturable: no allocation, no host-side control flow
 * that depends on device data; the update counter lives on the device, so a captured graph can be
 * replayed for every update. */
aframe_status aframe_stream_step(aframe_ctx* ctx, const float* d_new_samples, aframe_stream_state* st,
                                 float* d_scores, int32_t* d_n_scores);

/* ---- O-3..O-6 in one call: offline background analysis of a stored segment (C3) ---------
 * BASELINE.json configs[3]: the segment is whitened once per detector with the rolling-PSD rule
 * (aframe_whiten_rolling; output kept in the context's workspace as fp16 for the tensor-core path, else fp32),
 * then n_slides timeslides are scored: window i of slide k takes channel 0 (H1, held fixed) at whitened
 * index first + i*stride and every other channel at first + i*stride + slide_shifts[k] ("the Livingston
 * data is shifted in 1 s increments"; shifts in SAMPLES, applied to the whitened stream, C3).
 * Whitened index 0 is raw sample psd_len - stride - filter_len/2 of the segment.  Windows are scored
 * `batch` per launch sequence (configs[3]: 4096).  scores: [n_slides][n_windows] fp32 logits.
 * h_slide_shifts is a HOST array.  AFRAME_ESHAPE if any window reaches outside the whitened segment.
 *
 * aframe_score_timeslides      : d_strain / d_scores are DEVICE pointers; asynchronous on the stream.
 * aframe_score_timeslides_host : h_strain / h_scores are HOST pointers (pinned memory makes the copies
 *   asynchronous); the call copies the segment to the device, runs the same path, copies the scores back
 *   and synchronises the stream before returning. */
aframe_status aframe_score_timeslides(aframe_ctx* ctx, const aframe_weights* w, const float* d_strain,
                                      int64_t n_samples, int64_t ld, int64_t first, int64_t n_windows,
                                      const int64_t* h_slide_shifts, int32_t n_slides, int64_t batch,
                                      float* d_scores);
aframe_status aframe_score_timeslides_host(aframe_ctx* ctx, const aframe_weights* w, const float* h_strain,
                                           int64_t n_samples, int64_t ld, int64_t first, int64_t n_windows,
                                           const int64_t* h_slide_shifts, int32_t n_slides, int64_t batch,
                                           float* h_scores);

/* ---- NEXT-1  post-processing of the score series (readings D1-D3 of DESIGN.md) -------------------------
 * d_scores [n_series][ld] fp32 (e.g. the [n_slides][n_windows] output of aframe_score_timeslides), n valid per series.
 * d_integrated [n_series][n]: 1 s top hat = mean of the trailing n_int scores (n_int = inference rate x 1 s = 16;
 *   the first n_int - 1 entries average the scores that exist), float32 sums in index order.
 * Triggers: one per consecutive window of n_cluster integrated values (8 s = 128; a trailing partial window counts):
 *   d_trig_value [n_series][n_trig] = the maximum, d_trig_index [n_series][n_trig] = index of its first occurrence
 *   (a window that holds a NaN yields its first NaN: NaN propagates).
 *   *h_n_trig (HOST) = ceil(n / n_cluster).  The caller sizes the trigger arrays for that. */
aframe_status aframe_postprocess(aframe_ctx* ctx, const float* d_scores, int64_t n_series, int64_t n, int64_t ld,
                                 int32_t n_int, int32_t n_cluster, float* d_integrated, float* d_trig_value,
                                 int64_t* d_trig_index, int64_t* h_n_trig);

/* ---- how overlapping windows are planned (diagnostic; host arithmetic only, needs no device and no context) ------------
 * Windows taken in place at a spacing of window_spacing samples share every activation row that is out of reach of their own
 * zero padding: the tensor-core path runs each stage once over the stream of a launch sequence plus, per
 * window, the rows within reach of the padding.  This call reports that plan for a weight blob (version 1, as for
 * aframe_weights_load): *first_stage_blocks = basic blocks of the 64-channel stage run in shared form (0: none), then one
 * record per later stage in shared form.  In a packed stage, launched layer q computes per window one box of tbox[q] =
 * max(e_head[q], e_tail[q], 4) rows at each end (its edge rows), floor(128 / tbox[q]) boxes per 128-row MMA tile, in slots
 * of P rows: the box, the two rows next to the edge rows that later layers read (copied from the stream) and, if the next
 * stage is packed too, the rows its first two layers reach, which it reads in place (P is then even).  The last box of a half
 * may overhang into the spare_slots slots that follow.
 * AFRAME_EINVAL / AFRAME_ESHAPE for bad arguments or a bad table. */
typedef struct {
  int32_t first_layer, n_layers;   /* table index of the stage's entry conv; layers that launch (<= 16 are described) */
  int32_t T, C;                    /* rows per window and channels of the stage's output                             */
  int32_t head, tail;              /* rows at a window's start / end within reach of its zero padding, stage output  */
  int32_t packed;                  /* 1: packed edge batch; 0: fixed-length short windows                            */
  int32_t P;                       /* packed: rows per slot; else data rows of a short window                        */
  int32_t spare_slots;             /* packed: slots after each half                                                   */
  int32_t e_head[16], e_tail[16], tbox[16];
} aframe_stage_plan;
aframe_status aframe_describe_shared_plan(const void* host_blob, size_t bytes, int32_t kernel_len, int32_t n_channels,
                                          int32_t window_spacing, int64_t n_windows, int32_t* first_stage_blocks,
                                          aframe_stage_plan* stages, int32_t max_stages, int32_t* n_stages);

/* How many updates of this state were served by replaying the captured CUDA graph (0 for a context bound to the legacy
 * default stream, which cannot be captured, or while aframe_profile is on). */
int64_t aframe_stream_graph_replays(const aframe_stream_state* st);

/* 0 if this state runs one full forward of the window per update; else the number of CTAs of the cluster that runs the
 * incremental network ("snapshotting" taken through the network: windows of consecutive updates share every activation
 * row that is out of reach of their own zero padding, so an update computes, per layer, only stride / (samples per row) new
 * rows plus the window's first and last few rows -- at most 48 rows instead of 768 ... 96).  Used when cfg.precision is
 * AFRAME_F16 with a folded norm, the table is stem conv k7 s2 + ReLU + max-pool k3 s2 p1, k1 / k3 convs, head, cfg.stride is
 * a multiple of the network's total downsampling (32 for config-1) and at most 128, and cfg.stream_full_forward is 0.
 * Same roundings as the full forward (fp16 weights, one fp16 rounding per stored activation, fp32 accumulation), another
 * summation order: scores agree with it to ~1e-3 relative, not bit for bit. */
int32_t aframe_stream_incremental(const aframe_stream_state* st);

/* Host-only arithmetic (no CUDA call): rows the incremental network computes per update and layer for a weight blob and an
 * update stride.  For layer i of the blob's table (the head excluded): t_out[i] rows per window, of which the first
 * head_rows[i] and the last tail_rows[i] are within reach of the window's own zero padding (an output row is such a row iff
 * it reads padding or such a row of its input), and new_rows[i] = stride / (samples per row) rows enter per update.
 * *n_layers = 0 if the table or the stride does not qualify (see aframe_stream_incremental); arrays hold max_layers entries. */
aframe_status aframe_describe_stream_plan(const void* host_blob, size_t bytes, int32_t kernel_len, int32_t n_channels,
                                          int32_t stride, int32_t max_layers, int32_t* n_layers, int32_t* t_out,
                                          int32_t* head_rows, int32_t* tail_rows, int32_t* new_rows);

/* Number of kernels the library has launched on this context since creation (for bench accounting). */
int64_t aframe_launch_count(const aframe_ctx* ctx);

/* Multiply-accumulates the bf16 tensor-core convolutions (a-7) of this context have issued since creation: per launch,
 * (rows of all its MMA tiles, padding and separator rows included) x C_out x K.  Windows that overlap in time share the
 * interior rows of every stage, so this is less than the method's 1069.5 MMAC per window; bench.py
 * reports the tensor-core rate from this count, not from the algorithmic figure. */
double aframe_tensor_macs(const aframe_ctx* ctx);

/* ---- per-stage device timing (measurement aid) ------------------------------------------
 * aframe_profile(ctx, 1) clears the counters and makes every later call bracket each stage of the path
 * with a pair of CUDA events on the context's stream; aframe_profile(ctx, 0) stops.  aframe_profile_read
 * synchronises the stream and returns, per stage kind, the summed device time in milliseconds and the
 * number of kernel launches it covered (arrays of AFRAME_PROF_KINDS entries, HOST pointers). */
enum {
  AFRAME_PROF_WELCH = 0,    /* periodograms + PSD mean (a-2)            */
  AFRAME_PROF_DESIGN = 1,   /* whitening-filter design (a-3)            */
  AFRAME_PROF_WHITEN = 2,   /* overlap-save / FIR whitening (a-4)       */
  AFRAME_PROF_STEM = 3,     /* window assembly + stem + max-pool (a-5/6)*/
  AFRAME_PROF_CONV = 4,     /* residual-stage convolutions (a-7)        */
  AFRAME_PROF_HEAD = 5,     /* pool + linear head (a-8)                 */
  AFRAME_PROF_STREAM = 6,   /* ring-buffer bookkeeping (a-9)            */
  AFRAME_PROF_GATHER = 7,   /* shared stages: edge-batch gathers, stitch, head-rows sum (a-7 bookkeeping) */
  AFRAME_PROF_KINDS = 8
};
aframe_status aframe_profile(aframe_ctx* ctx, int enable);
/* One forward pass of aframe_forward on d_windows [B][C][kernel_len] with a CUDA-event pair around every layer's
 * launch (bf16 path; B at most one internal chunk).  h_ms: HOST array of n_layers floats (layer-table order; the stem's
 * conv + max-pool are reported on entry 0, the head on the last entry).  Synchronises. */
aframe_status aframe_profile_layers(aframe_ctx* ctx, const aframe_weights* w, const float* d_windows, int64_t B,
                                    float* d_scores, float* h_ms, int32_t n_layers);
aframe_status aframe_profile_read(aframe_ctx* ctx, double* h_ms, int64_t* h_launches);

#ifdef __cplusplus
}
#endif
#endif /* AFRAME_H_ */
