/*
 * gwstream.h -- C ABI of the B200-native streaming inference engine for the hot path of
 * arXiv:2108.12430 ("Hardware-accelerated Inference for Real-Time Gravitational-Wave Astronomy").
 *
 * The interface follows the paper's statement of the problem (section B.1):
 *   "Inference requests are made to this model providing a floor(fs/r)-sized stream of strictly
 *    new samples that are used to update the state to a new snapshot, which is then passed to
 *    downstream static models."
 * and the ensemble order of PAPER.md:76 (Fig. 4) / :212: snapshotter -> one DeepClean per detector
 * -> aggregation + subtraction -> BBHnet on the cleaned strain of both detectors.
 *
 * Conventions
 *  - Plain C, opaque handles, no exceptions.  Every call returns 0 (GW_OK) or a negative code;
 *    gw_last_error(handle) returns the description of the last failure of a call on that handle
 *    (gw_last_error(NULL): of the last failed call on this thread, e.g. a create that returned no handle).
 *  - No process-global switches: everything that selects a code path is a field of gw_options, fixed
 *    when a handle is created.
 *  - "dev" pointers are CUDA device pointers on the current device, "host" pointers are host
 *    memory.  The caller owns every buffer it passes; the engine owns all persistent state (rings,
 *    overlap-add accumulators, activations, weights -- parameters are COPIED at create time).
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is
 *    enqueued on it and is asynchronous unless stated.  One handle is used from one host thread at
 *    a time, and by one CUDA stream at a time.
 *  - Per update the calls must come in this order:
 *        gw_stream_update -> gw_deepclean_forward -> gw_cleaned_strain -> gw_bbh_score
 *    (or one gw_step).  Anything else returns GW_ESTATE.  Results of update t are a pure function
 *    of all samples through update t.
 *  - There is no CPU fallback: without a CUDA device every compute call returns GW_ECUDA.
 *
 * Layouts are row-major with the last index fastest, written [a][b][c].
 * n = n_streams, C = channels, W = window, S = stride (both in samples), D = detectors.
 */
#ifndef GWSTREAM_H
#define GWSTREAM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { GW_OK = 0, GW_EINVAL = -1, GW_ESTATE = -2, GW_ENOMEM = -3, GW_ECUDA = -4 };
enum { GW_BF16 = 0, GW_FP16 = 1 };                       /* storage/multiply type; accumulation is fp32 */
enum { GW_CONV = 0, GW_CONVT = 1 };                      /* Conv1d | ConvTranspose1d */
enum { GW_ACT_NONE = 0, GW_ACT_TANH = 1, GW_ACT_RELU = 2 };
enum { GW_FINAL = 0, GW_RUNNING = 1 };                   /* gw_cleaned_strain output selection */
enum { GW_AGG_HANN_OLA = 0, GW_AGG_LAST_STRIDE = 1 };    /* aggregation of overlapping predictions */
enum { GW_IMPL_UMMA = 0, GW_IMPL_SIMT = 1 };             /* conv GEMM implementation (SIMT = debug cross-check) */

typedef struct gw_stream gw_stream;
typedef struct gw_deepclean gw_deepclean;
typedef struct gw_bbh gw_bbh;
typedef struct gw_pipeline gw_pipeline;
typedef struct gw_offline gw_offline;

/* One convolution layer, parameters in HOST memory, fp32, unfolded.
 *  kind GW_CONV : y[co][l] = b[co] + sum_ci sum_j w[co][ci][j] x[ci][stride*l + j - pad_l], zero
 *                 padding pad_l / pad_r; w is [cout][cin][k].
 *  kind GW_CONVT: the adjoint, y[co][m] = b[co] + sum_ci sum_{l,j: stride*l + j - pad_l = m}
 *                 w[ci][co][j] x[ci][l]; pad_l = padding, pad_r = output_padding; w is [cin][cout][k].
 *  BatchNorm (inference): if bn_gamma != NULL, z -> gamma (z - mean)/sqrt(var + eps) + beta is
 *  applied between the convolution and the activation; it is folded into w and b in double
 *  precision at create time (BASELINE.json configs[1]: "folded BatchNorm").
 *  pool: MaxPool1d(pool, stride pool) after the activation (1 = none).
 *  Supported by the tensor-core path: GW_CONV with k odd, stride 2, pad_l = pad_r = k/2 (DeepClean
 *  encoder); GW_CONVT with k odd, stride 2, pad_l = k/2, pad_r = 1 (decoder); GW_CONV with stride 1,
 *  pad_l + pad_r = k - 1, pool 4 (classifier).  Other shapes return GW_EINVAL. */
typedef struct {
    int kind, cin, cout, k, stride, pad_l, pad_r, act, pool;
    const float *w, *b;
    const float *bn_gamma, *bn_beta, *bn_mean, *bn_var;
    float bn_eps;
} gw_conv_layer;

/* DeepClean stage: one network PER DETECTOR ("two DeepClean instances").
 *  layers[d*n_layers + i] is layer i of detector d; the last layer must have cout = 1.
 *  witness_rows[d*n_witness + c] / strain_row[d]: rows of the snapshot ring (one
 *  snapshotter holds all data sources and hands slices to each model).
 *  agg: GW_AGG_HANN_OLA (periodic-Hann overlap-add normalised by the summed window; needs
 *  window % stride == 0 and window/stride >= 2) or GW_AGG_LAST_STRIDE (each
 *  prediction keeps only its most recent `stride` samples).
 *  delta: aggregation-latency offset in samples: the classifier window and the
 *  LAST_STRIDE span end `delta` samples before the newest sample.  0 <= delta <= window - stride. */
typedef struct {
    int n_det, n_layers, n_witness;
    const gw_conv_layer *layers;
    const int *witness_rows;
    const int *strain_row;
    int agg, delta;
} gw_dc_spec;

/* BBH classifier: conv blocks (conv -> ReLU -> max-pool) on the D cleaned
 * strains, global average pooling, dense layers (ReLU between, none after the last), sigmoid.
 *  dense_w[i] is [dense_dims[i+1]][dense_dims[i]] fp32 host, dense_b[i] is [dense_dims[i+1]];
 *  dense_dims[0] = cout of the last conv, dense_dims[n_dense] = 1.  n_dense must be 2.
 *  length: classifier window L_b in samples (multiple of 64, <= 4096 and <= window). */
typedef struct {
    int n_convs;
    const gw_conv_layer *convs;
    int n_dense;
    const int *dense_dims;
    const float *const *dense_w;
    const float *const *dense_b;
    int length;
} gw_bbh_spec;

/* Options fixed at create time (pass NULL for the defaults).  None of them changes WHAT is computed:
 *  conv_impl   GW_IMPL_UMMA (default): tcgen05/TMEM/TMA conv GEMMs.  GW_IMPL_SIMT: a slow CUDA-core kernel over the
 *              same operand layout, kept to bisect tensor-core bugs in tests.  Both are CUDA; neither is a fallback.
 *  fuse_tail   1 (default): the last tensor-core layer of DeepClean (ConvTranspose1d -> <= 32 channels, tanh) and the
 *              final 1-channel ConvTranspose1d (k = 7) run as one kernel; the activation between them is never stored
 *              (gw_deepclean_activation returns GW_ESTATE for it).  0: it is written to HBM.  Agree within rounding.
 *  pdl         1 (default): programmatic dependent launch between the kernels of an update (each kernel's prologue
 *              overlaps its predecessor's tail; it waits on the device before touching the predecessor's output).
 *  snake       1 (default): consecutive DeepClean layers walk their (window, tile) list in alternating directions, so a
 *              layer starts on the activations its predecessor wrote last (still in L2).
 *  two_sm      1 (default): CTA-pair kernel (tcgen05 cta_group::2, M = 256) for the layers whose weights do not fit in
 *              shared memory (GEMM N = 256).
 *  skip_zeros  1 (default): the resident-weight conv GEMMs skip the K steps and halves of N that no filter tap reaches.
 *  pdl / snake / two_sm / skip_zeros are scheduling only (or skip exact zeros): results are BIT-identical either way.
 *  incremental 0 (default): every update recomputes the whole window.  1: the exact incremental path (D13,
 *              only floor(fs/r) samples are new per update): every layer's activations live
 *              in a ring over absolute position and an update recomputes only the rows whose receptive field reaches
 *              the new samples or one of the two window edges; every other row IS the previous update's value.
 *              Results are bit-identical to full recomputation.  Needs stride and window to be multiples of
 *              2^(encoder depth), window a multiple of 128 * 2^(encoder depth), the fused tail and GW_IMPL_UMMA
 *              (GW_EINVAL otherwise).
 *  fuse_bbh    1 (default): the whole classifier (three conv blocks, pooling, dense head, sigmoid) runs as ONE kernel
 *              with one CTA per window and every activation in shared memory, when its shape is three blocks of k = 8,
 *              pad_l = 3 with at most 32 / 64 and exactly 128 output channels, at most 2 detectors, a window that is a
 *              multiple of 512 in [512, 4096] and a dense hidden width <= 64 (BASELINE.json configs[2]); other shapes,
 *              fuse_bbh = 0 and GW_IMPL_SIMT take the three-kernel path (first block on CUDA cores, blocks 2 and 3 as
 *              conv GEMMs with activations in global memory).  Both paths keep the fp32 input unrounded; they agree
 *              within rounding (different summation order).
 *  fuse_head   1 (default): the first two DeepClean layers (stride-2 Conv1d -> 32 and -> 64 channels, tanh) run as one
 *              kernel: two tiles of layer 0 are activated into shared memory as one operand tile of layer 1, a second
 *              chain of tcgen05.mma produces layer 1's rows, and layer 0's activation is never written (or read back) --
 *              a quarter of the two layers' HBM traffic (gw_deepclean_activation returns GW_ESTATE for layer 0).  Whole
 *              windows only (not with `incremental`), GW_IMPL_UMMA.  The same products in the same order: BIT-identical
 *              to fuse_head = 0. */
typedef struct {
    int conv_impl, fuse_tail, pdl, snake, two_sm, skip_zeros, incremental, fuse_bbh, fuse_head;
} gw_options;
void gw_options_default(gw_options *o);

/* Description of the last failure on `handle` (any gw_* handle), or with NULL of the last failed call on the calling
 * thread.  The string is owned by the library and valid until the next failing call on that handle / thread. */
const char *gw_last_error(const void *handle);

/* Number of CUDA kernels this library has launched (or captured into a graph and replayed) on
 * behalf of the calling process so far (atomic counter); used by bench.py for "gpu_launches". */
int64_t gw_kernel_launches(void);

/* ---- snapshotter -------------------------------------------------------------
 * gw_stream_create: zeroed ring state [n][C][W] fp32 on the current device, sample counter 0.
 *   Requires n >= 1, C >= 1, fs >= 1, 1 <= S <= W.
 * gw_stream_update: new_samples_dev is [n][C][S] fp32, strictly new samples; appends them and
 *   advances the counter by S.  128-bit path when S % 4 == 0 and W % 4 == 0, scalar otherwise.
 * gw_stream_snapshot (test hook): writes the time-ordered snapshot [n][C][W] to out_dev and, if
 *   first_index_host != NULL, the absolute index (t+1)S - W of its first sample (negative during
 *   warm-up; samples before the stream start read as 0).  Synchronises `stream`.
 * gw_stream_count: samples per channel appended so far (host-side mirror of the device counter). */
int gw_stream_create(gw_stream **out, int n_streams, int channels, int fs, int window, int stride);
int gw_stream_destroy(gw_stream *s);
int gw_stream_update(gw_stream *s, const float *new_samples_dev, void *stream);
int gw_stream_snapshot(gw_stream *s, float *out_dev, int64_t *first_index_host, void *stream);
int64_t gw_stream_count(const gw_stream *s);

/* ---- DeepClean ------------------------------------------------------------------
 * gw_deepclean_create: folds BatchNorm, rounds weights RN-even to `dtype`, builds the GEMM
 *   operands and TMA descriptors, allocates activations and aggregation state.  The stream must
 *   outlive the handle.  Must be created before the stream's first update.
 * gw_deepclean_forward: gathers the current window of every (stream, detector), converts it to
 *   `dtype` channels-last, runs all layers; the raw prediction p_t [n][D][W] fp32 stays inside.
 * gw_deepclean_noise (test hook): copies p_t to out_dev [n][D][W].
 * gw_cleaned_strain: aggregates p_t into the running noise estimate (Hann overlap-add + window
 *   normalisation, or LAST_STRIDE), subtracts it from the strain and writes to out_dev
 *   (may be NULL):  GW_FINAL   -> [n][D][S], the S samples that became final with this update
 *                                 (absolute index (t+1)S - W ...; LAST_STRIDE: (t+1)S - S - delta ...)
 *                   GW_RUNNING -> [n][D][W], the running-normalised cleaned window.
 *   Samples with negative absolute index are written as 0.
 * gw_noise_estimate (test hook): the running noise estimate nhat over the current window,
 *   [n][D][W] (0 where no prediction covers the sample).  Valid after gw_cleaned_strain. */
int gw_deepclean_create(gw_deepclean **out, gw_stream *s, const gw_dc_spec *spec, int dtype, const gw_options *opts);
int gw_deepclean_destroy(gw_deepclean *dc);
int gw_deepclean_forward(gw_deepclean *dc, void *stream);
int gw_deepclean_noise(gw_deepclean *dc, float *out_dev, void *stream);
int gw_cleaned_strain(gw_deepclean *dc, float *out_dev, int mode, void *stream);
int gw_noise_estimate(gw_deepclean *dc, float *out_dev, void *stream);
/* test hook: copy the activations after layer `layer` (0-based) as stored, 16-bit channels-last
 * [n][D][L_layer][C_padded]; *rows / *cols (host, may be NULL) receive L_layer and C_padded. */
int gw_deepclean_activation(gw_deepclean *dc, int layer, void *out_dev, int64_t out_bytes,
                            int *rows, int *cols, void *stream);

/* ---- BBH classifier ---------------------------------------------------------------
 * gw_bbh_create: dc may be NULL for a stateless batch classifier (gw_bbh_score_batch only), in
 *   which case n_det detectors and max_batch windows are assumed.
 * gw_bbh_score: scores_dev [n] fp32 in (0,1), on the window
 *   [(t+1)S - delta - L_b, (t+1)S - delta) of the running cleaned strain of this update.
 * gw_bbh_score_batch: stateless; windows_dev [B][D][L_b] fp32, scores_dev [B]; B <= max_batch. */
int gw_bbh_create(gw_bbh **out, gw_deepclean *dc, const gw_bbh_spec *spec, int dtype, int n_det,
                  int max_batch, const gw_options *opts);
int gw_bbh_destroy(gw_bbh *b);
int gw_bbh_score(gw_bbh *b, float *scores_dev, void *stream);
int gw_bbh_score_batch(gw_bbh *b, const float *windows_dev, int batch, float *scores_dev, void *stream);

/* ---- one update as one CUDA-graph replay (north_star (5)) ----------------------------------------
 * gw_pipeline_create: ties the three stages (bbh may be NULL).  The first gw_step captures
 *   update -> forward -> cleaned(GW_FINAL) -> score into a CUDA graph; later steps replay it (the ring
 *   head lives in device memory, so the graph is replayed unchanged).
 * gw_step: device buffers.  new_samples_dev [n][C][S]; scores_dev [n] (ignored without bbh);
 *   cleaned_final_dev [n][D][S].  The pointers are parameters of graph nodes: passing different buffers from one
 *   call to the next (rotating output buffers, say) is a node-parameter update of the instantiated graph, never a
 *   re-capture.  `stream` must not be the legacy default stream.
 * gw_step_host: HOST buffers; copies new samples host->device, replays the graph, copies scores
 *   and final cleaned samples device->host, and synchronises.  Pinned host memory makes the copies
 *   asynchronous; pageable memory works but is slower. */
int gw_pipeline_create(gw_pipeline **out, gw_stream *s, gw_deepclean *dc, gw_bbh *bbh);
int gw_pipeline_destroy(gw_pipeline *p);
int gw_step(gw_pipeline *p, const float *new_samples_dev, float *scores_dev, float *cleaned_final_dev,
            void *stream);
int gw_step_host(gw_pipeline *p, const float *new_samples_host, float *scores_host,
                 float *cleaned_final_host, void *stream);
/* gw_step_host_async: the throughput form of gw_step_host (offline regime).  Same arguments; does
 * NOT synchronise.  The host->device copy of this call's samples runs on an internal copy stream into one of two
 * staging buffers and overlaps the previous step's kernels; scores and final cleaned samples reach the host
 * buffers in stream order on `stream` (pinned, mapped buffers are written by the kernels themselves; pageable ones
 * through copies).  Every host buffer passed to a call must stay valid (and, for the outputs, unread)
 * until `stream` has been synchronised past that call.  Use pinned host memory. */
int gw_step_host_async(gw_pipeline *p, const float *new_samples_host, float *scores_host,
                       float *cleaned_final_host, void *stream);
/* number of kernel nodes in the captured graph (0 before the first gw_step) */
int gw_pipeline_graph_nodes(const gw_pipeline *p);

/* ---- pre/post-processing at the edges of DeepClean (PAPER.md:198 "preprocesses", :212 "postprocessed"; the paper
 * does not define them: reading A14 of DESIGN.md fixes per-channel standardisation) -------------------------------
 * Witness c of detector d enters the network as (x - wit_mean[d*n_witness+c]) / wit_std[...] (applied in fp32
 * when the sample is converted to the 16-bit storage type), and the aggregated estimate is subtracted from the
 * strain as strain_std[d] * nhat + strain_mean[d] (gw_noise_estimate returns the rescaled estimate; the raw
 * predictions of gw_deepclean_noise are unscaled).  Host arrays, copied; a NULL array means identity for that part;
 * the default is identity everywhere, which is bit-exact with no processing at all.  wit_std must be > 0.
 * gw_deepclean_set_scaling must precede the first update (GW_ESTATE otherwise: the state holds converted samples). */
int gw_deepclean_set_scaling(gw_deepclean *dc, const float *wit_mean, const float *wit_std, const float *strain_mean,
                             const float *strain_std);
int gw_offline_set_scaling(gw_offline *o, const float *wit_mean, const float *wit_std, const float *strain_mean,
                           const float *strain_std);

/* Band-limiting of the predicted noise and whitening of the classifier input ("the noise frame ... is
 * postprocessed then subtracted from the associated strain", :212 "the cleaned strains are combined and postprocessed
 * then passed to BBHnet"; the paper defines neither operation: DESIGN.md D11, D12 fix them as causal FIR filters whose
 * taps the caller supplies -- a band-pass for D11, a whitening filter for D12).
 * gw_deepclean_set_postfilter (D11): the STREAM of emitted estimate samples e[a] (HANN_OLA: the samples that become
 *   final, LAST_STRIDE: the kept stride; unscaled, 0 before the stream start) is filtered causally with state carried
 *   from update to update, e~[a] = sum_{j < n_taps} taps[j] e[a - j], and the final cleaned samples (GW_FINAL,
 *   gw_step's cleaned_final) become strain - (strain_std * e~ + strain_mean).  Running values (GW_RUNNING,
 *   gw_noise_estimate, the classifier input) are provisional values inside the window and are not filtered.
 *   taps_host: [n_taps] host floats, copied; 1 <= n_taps <= 64 and n_taps - 1 <= stride; NULL or 0 taps switches it off;
 *   taps = {1} is a bit-exact no-op.  Before the first update (GW_ESTATE otherwise).
 * gw_bbh_set_whitening (D12): the classifier sees y_d[i] = sum_{j < n_taps} taps[d][j] x_d[i - j], x_d[i < 0] = 0 (zero
 *   initial state at the start of the classifier window), for gw_bbh_score, gw_bbh_score_batch and gw_step alike.
 *   taps_host: [n_det][n_taps], copied; 1 <= n_taps <= 64; NULL or 0 switches it off.  Call it before the first
 *   gw_step (a captured graph keeps the setting it was captured with). */
int gw_deepclean_set_postfilter(gw_deepclean *dc, const float *taps_host, int n_taps);
int gw_bbh_set_whitening(gw_bbh *b, const float *taps_host, int n_taps);

/* ---- offline / non-streaming mode (PAPER.md:174 "adjacent frames ... in parallel", :202 offline regime, :216
 * non-streaming ensemble; D9) ---------------------------------------------------
 * One launch sequence cleans an ARCHIVAL segment of ONE stream: T = window + (n_windows - 1) * stride samples per
 * channel are cut into the n_windows windows [j*stride, j*stride + window) (the streaming path's window grid
 * without its warm-up windows), every window goes through DeepClean (same kernels as the streaming path, the
 * windows folded into the GEMM M dimension), and the predictions are combined by the periodic-Hann overlap-add
 * normalised by the summed weights of the windows that actually cover a sample; cleaned = strain - estimate.
 * A sample covered by all window/stride windows is bit-identical to the streaming path's final value.
 * gw_offline_create: spec as for gw_deepclean_create (agg and delta are ignored); window % stride == 0,
 *   window/stride >= 2.  Owns all device state.  Errors: GW_EINVAL, GW_ENOMEM, GW_ECUDA.
 * gw_offline_samples: T.
 * gw_offline_run: samples_dev [channels][T] fp32, cleaned_dev [n_det][T] fp32, noise_dev [n_det][T] or NULL (the
 *   estimate that was subtracted), all device pointers owned by the caller; asynchronous on `stream`.
 * gw_offline_predictions (test hook): raw per-window predictions [n_windows][n_det][window] of the last run. */
int gw_offline_create(gw_offline **out, const gw_dc_spec *spec, int channels, int fs, int window, int stride,
                      int n_windows, int dtype, const gw_options *opts);
int gw_offline_destroy(gw_offline *o);
int64_t gw_offline_samples(const gw_offline *o);
int gw_offline_run(gw_offline *o, const float *samples_dev, float *cleaned_dev, float *noise_dev, void *stream);
int gw_offline_predictions(gw_offline *o, float *out_dev, void *stream);

/* ---- The entry point that allocates nothing (csrc/gw_noalloc.cu) -------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the offline overlap-add above (D9) on per-window predictions the caller
 * already holds, with no handle and no allocation.  It calls no cudaMalloc, cudaFree or allocating library routine: the
 * Hann window and the summed-weight table it needs live in a fixed __device__ array inside the library (640 KiB, held by
 * every GPU that loads the library until the process exits), whose device address is looked up once per device on the
 * first call made with that device current.
 *   pred_dev    [n_windows][n_det][window] fp32, window j = samples [j*stride, j*stride + window) of the segment
 *   strain_dev  [n_det][T] fp32, T = window + (n_windows - 1) * stride
 *   cleaned_dev [n_det][T] fp32 out: strain - estimate;  noise_dev [n_det][T] out or NULL: the estimate
 *   post_dev    [n_det][2] fp32 (scale, offset) applied to the normalised estimate, or NULL for (1, 0)
 * All are device pointers owned by the caller, none may alias an output.  Asynchronous on `stream` (three kernels).
 * Same arithmetic as gw_offline_run's overlap-add (tables computed on the device instead of the host).
 * Limits: window <= GW_OLA_NOALLOC_MAX_WINDOW, window % stride == 0, window / stride >= 2, n_det <= 65535; anything
 * else returns GW_EINVAL and launches nothing.  GW_ECUDA: no device / launch failure (there is no CPU fallback).
 * The scratch array is shared by all calls on a device and keeps the last call's tables; every call rewrites what it
 * reads.  Calls on one stream are ordered; calls that OVERLAP on the GPU (different streams or threads) race on it
 * unless they use the same (window, stride). */
#define GW_OLA_NOALLOC_MAX_WINDOW 32768
int gw_ola_offline_noalloc(const float *pred_dev, const float *strain_dev, float *cleaned_dev, float *noise_dev,
                           const float *post_dev, int n_windows, int n_det, int window, int stride, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* GWSTREAM_H */
