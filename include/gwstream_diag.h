/*
 * gwstream_diag.h -- measurement and diagnostic entry points of libgwstream.so.  NOT part of the product interface
 * (include/gwstream.h): bench.py and the tests use them to time the kernels of a step and to reproduce the
 * micro-benchmark behind the shared-memory operand roofline.  Same conventions as gwstream.h.
 */
#ifndef GWSTREAM_DIAG_H
#define GWSTREAM_DIAG_H

#include "gwstream.h"

#ifdef __cplusplus
extern "C" {
#endif

/* gw_step_profile: ONE update through a CUDA graph of exactly the kernels gw_step replays (same launch attributes,
 * programmatic dependent launch included), in which every kernel additionally stamps %globaltimer when its first CTA
 * starts and when its last CTA has finished; synchronises `stream`.  Counts as one update of the stream.
 *  begin_us[i], end_us[i] (host, i < min(*n_out, max_kernels)): start and end of kernel i in microseconds relative to
 *  the start of the step's first kernel.  Kernels overlap under PDL (a successor's prologue runs under its
 *  predecessor's tail), so the decomposition of the step is excl_i = end_i - max(begin_i, end_{i-1}); their sum is
 *  the span of the step on the device and cannot exceed the step time measured around the graph launch.
 *  sm_mhz[i] (host, may be NULL): the SM clock kernel i actually ran at = the kernel's length in SM cycles (clock64 of its
 *  CTA 0) over its length in ns (%globaltimer of the same CTA).  nvidia-smi samples every 25 ms at best; a kernel lasts
 *  0.01-0.2 ms and the power cap moves the clock from one kernel to the next.
 *  gw_profile_label(p, i): kernel i's name ("snapshot_append", "gemm.dc0", ... "aggregate", "bbh_fused" -- or, as three
 *  kernels, "bbh_conv1", "gemm.bbh1", "gemm.bbh2").
 *  gw_profile_flops(p, i): algorithmic FLOPs kernel i EXECUTED in that step (real channels and taps only, whole
 *  batch; with gw_options.incremental: the rows of the tiles that were recomputed); 0 for non-GEMM kernels.
 *  gw_profile_smem_bytes(p, i): shared-memory traffic of conv GEMM kernel i by the accounting of DESIGN.md section 7
 *  (MMA operand reads + TMA fills + epilogue staging, all SMs); 0 for other kernels. */
int gw_step_profile(gw_pipeline *p, const float *new_samples_dev, float *scores_dev, float *cleaned_final_dev,
                    void *stream, int max_kernels, double *begin_us, double *end_us, double *sm_mhz, int *n_out);
const char *gw_profile_label(const gw_pipeline *p, int i);
double gw_profile_flops(const gw_pipeline *p, int i);
double gw_profile_smem_bytes(const gw_pipeline *p, int i);

/* Measured cycles per tcgen05.mma (cta_group::1, kind::f16, M = 128, K = 16, both operands in shared memory,
 * SWIZZLE_128B) for GEMM N in {16, 32, 64, 128, 256} on the current device: one CTA issues 1024 MMAs back to back with
 * a conv layer's descriptor pattern.  *issue_cycles = issue-loop time per MMA, *complete_cycles = time until the last
 * one has retired, per MMA (host pointers).  Synchronises the device. */
int gw_probe_mma_cycles(int N, float *issue_cycles, float *complete_cycles);

/* Measured rate of the DeepClean epilogues' activation instruction on the current device, in results per clock per SM
 * (host pointer), with `threads` threads per SM (multiple of 32, <= 1024) running eight independent chains each:
 * mode 0 tanh.approx.f32 (fp16 engine: one MUFU operation per tanh), 1 tanh.approx.f16x2 (two results per instruction --
 * and two MUFU operations: no gain), 2 ex2.approx + rcp.approx (bf16 engine's exact tanh: *result counts tanh evaluations,
 * two MUFU operations each).  The MUFU pipe is the second floor under the thin conv layers: a layer
 * evaluates rows x channels tanh per window.  Synchronises the device. */
int gw_probe_mufu_rate(int mode, int threads, float *results_per_clock_per_sm);

/* The arithmetic behind gw_options.incremental (D13), host only: for a stack of stride-2 layers
 * (kind, k as in gw_conv_layer; weights are not read) and `stride` new samples per update, left[i] / right[i] = how
 * many OUTPUT positions of layer i at the left / right end of the window differ from the previous update's value at
 * the same absolute position (receptive field reaches the zero-padded window edge, or the new samples).  The engine
 * recomputes those rows (rounded up to tiles) and keeps every other row.  tests/test_oracle_pins.py checks the numbers
 * against the oracle run on two overlapping windows. */
int gw_incremental_zones(const gw_conv_layer *layers, int n_layers, int stride, int *left, int *right);

/* Host only (no CUDA device needed): the tensor-core operand images of the one-kernel classifier (gw_options.fuse_bbh)
 * exactly as gw_bbh_create uploads them, so that their construction can be checked without a GPU.  All three are
 * K-major SWIZZLE_128B matrices of 16-bit storage values (rows of 64 values = 128 bytes; the 16-byte chunk c of row r sits
 * at chunk c ^ (r & 7)):
 *   w1 [128 rows][64]:           row = phase q * 32 + cout, k = (cin * 2 + part) * 16 + i holds tap j = i - q of
 *                                w[cout][cin][.] (i = 0..10: input sample 4r - 3 + i of im2col row r; part 0 multiplies
 *                                the 16-bit head of a sample, part 1 what that rounding lost) -- block 1 as a Toeplitz matrix;
 *   w2 [4 tap pairs][64 rows][64]:  block j / 2, row = cout, k = (j & 1) * 32 + cin;
 *   w3 [8 taps][128 rows][64]:      block j, row = cout, k = cin.
 * Sizes in 16-bit values: 8192, 16384, 65536.  GW_EINVAL if the spec is not a shape that kernel takes (gwstream.h,
 * gw_options.fuse_bbh). */
int gw_bbh_fused_images(const gw_bbh_spec *spec, int dtype, uint16_t *w1, uint16_t *w2, uint16_t *w3);

#ifdef __cplusplus
}
#endif
#endif /* GWSTREAM_DIAG_H */
