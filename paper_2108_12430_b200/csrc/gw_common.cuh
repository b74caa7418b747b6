// gw_common.cuh -- shared declarations of the CUDA path (engine-internal, not part of the ABI).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gw {

constexpr int kMaxSeg = 48;        // K segments (64 elements each) per conv GEMM
constexpr int kTileM = 128;        // UMMA M: one TMEM lane per output row
constexpr int kSegK = 64;          // 64 x 16-bit = one 128-byte swizzle row

enum { FMT_FP16 = 0, FMT_BF16 = 1 };                       // UMMA instruction-descriptor encoding
enum { EPI_STORE = 0, EPI_POOL = 1, EPI_POOL_HEAD = 2, EPI_FINAL = 3, EPI_CHAIN = 4 };
enum { ACT_NONE = 0, ACT_TANH = 1, ACT_RELU = 2 };

constexpr int kMaxCb = 8;          // 64-column blocks of the A view (a_cols <= 512)
constexpr int kMaxShift = 6;       // distinct row shifts of one layer

// One convolution layer expressed as
//     D[m][n] = sum over segments (cb, a):  A[m + a][64 cb .. 64 cb + 64) . B[n][64 s .. 64 s + 64),  s = seg_of[cb][a - a_min]
// where A is a 2-D view [rows][cols] of a channels-last activation tensor per batch item (rows out of
// range read as zero = the layer's zero padding) and B is the per-detector weight matrix whose K order
// is the segment order (cb outer, shift inner).
struct ConvGemmParams {
    CUtensorMap tmA;               // 3-D (cols, rows, batch), box (64, slab_rows, 1), SWIZZLE_128B
    CUtensorMap tmB;               // 3-D (K = 64 n_seg, N, n_det), box (64, N, 1), SWIZZLE_128B
    CUtensorMap tmOut;             // EPI_STORE: 3-D (N, M, batch), box (min(N, 64), 32, 1), swizzle = box row (128B / 64B)
    const void* A;                 // raw pointers of the same operands (SIMT cross-check kernel)
    const void* B;
    int a_rows, a_cols;            // A view per batch item (logical rows: out-of-range rows read as zero)
    int a_rows_tm;                 // rows per batch item of the underlying tensor (= a_rows, or 2 a_rows for a mirror ring)
    // Mirror-ring source (first DeepClean layer): the window is rows [off, off + a_rows) of a ring that holds
    // every sample twice (slots i and i + W), off = (*a_count mod a_ring_W) / a_ring_div, read on the device so
    // that a captured graph replays unchanged.  Rows outside [0, a_rows) are zeroed in shared memory after the
    // TMA load (the ring holds real samples there, not padding).  a_count == nullptr: plain activation tensor.
    const long long* a_count;
    // Offline source (a_4d = 1): tmA is 4-D (cols, rows, detector, window) over ONE stream's 16-bit segment
    // [n_det][T][cpad]; window j is the overlapping row range starting S/2 rows after window j-1 (its stride in the
    // tensor map), so no per-window copy exists and rows outside [0, a_rows) are still TMA's zero fill.
    int a_4d;
    int a_ring_W, a_ring_div;
    int M;                         // output rows per batch item
    int N;                         // GEMM N, multiple of 32, <= 256
    int n_seg;
    int n_det;                     // weight set = batch % n_det
    int fmt;                       // FMT_*
    int epi, act;
    int n_cb, a_min, n_shift;      // column blocks, first row shift, number of row shifts
    int slab_rows;                 // 128 + n_shift - 1: rows of A one output tile needs
    int b_resident;                // 1: all of B lives in shared memory for the CTA's lifetime
    int sa_stages, sb_stages;      // A-slab ring depth, B ring depth (streaming mode)
    int out_bufs;                  // EPI_STORE: output staging buffers per epilogue warp (1 or 2)
    int tiles_m;                   // output tiles per batch item: ceil(M / tile_stride)
    // Tile t covers output rows [t * tile_stride + tile_row0, ... + 128).  128 / 0 everywhere except
    // EPI_FINAL, whose tiles overlap by one halo row on each side (126 / -1).
    int tile_stride, tile_row0;
    // 1: walk the (batch item, tile) work list backwards.  Consecutive layers alternate direction, so a
    // layer starts on the activations its predecessor wrote LAST -- the part still resident in the 126 MB L2.
    int reverse;
    // EPI_STORE: tiles per accumulator stage (0 = as many as fit: 256 / N).  The plan lowers it when the launch has too
    // few stages' worth of work to fill the persistent CTAs evenly (small stream counts: latency, wave quantisation).
    int g_tiles;
    int two_sm;                    // 1: CTA-pair kernel (tcgen05 cta_group::2, M = 256), chosen by conv_gemm_plan
    // Incremental path (gw_options.incremental, D13).  The OUTPUT is a mirror ring as well: tmOut spans
    // 2 * M rows per batch item, the current window starts at row out_off = (*a_count mod a_ring_W) / out_ring_div and
    // every row is stored twice (rows r and r +- M), so that the consumer's window is contiguous.  0: plain tensor.
    int out_ring_div;
    // Work list per batch item: v_tiles "virtual" tiles, of which the first v_left are tiles 0 .. v_left-1 (rows whose
    // receptive field reaches the LEFT window edge) and the rest are the LAST v_tiles - v_left tiles (rows that see the
    // new samples or the right window edge).  Full recomputation: v_tiles = v_left = tiles_m.
    int v_tiles, v_left;
    // Zone launches, EPI_STORE: the recomputed rows are the first z_left and the last z_right rows of the layer; an epilogue
    // warp whose 32-row quadrant of a tile holds none of them skips it (the ring keeps those rows' values, which ARE the
    // values the tile would store again).  0 / 0: every row is live.
    int z_left, z_right;
    int pred_ring;                 // EPI_FINAL: pred is a ring over absolute sample index mod 4 M (no mirror: row stores)
    // CTA-pair kernel on a ring input: one tensor map PER WINDOW HEAD (device array of a_ring_W / head_div maps, the
    // map of head h based at the ring row where that window starts and a_rows rows tall), so that rows outside the
    // window are TMA's zero fill exactly as for a plain activation tensor -- no zeroing in shared memory, which the
    // pair kernel (the peer's slab is consumed by the leader's MMAs) has no warp in the right place for.
    const CUtensorMap* tmA_heads;
    int head_div;                  // head index = (*a_count mod a_ring_W) / head_div  (= the stride S)
    // CTA-pair kernel, zones packed (k_conv_gemm_2sm): a tile holds pk_k consecutive batch items, one segment of
    // pk_nl + pk_nr rows each.  Inside a segment the left zone's pk_left output rows are rows [0, pk_left) and read slab
    // rows [0, pk_nl) (loaded through tmA_heads_left: the per-head maps with a box of pk_nl rows, pk_nl = pk_left +
    // n_shift - 1 rounded up to 8); the right zone's pk_right rows are rows [pk_nl, pk_nl + pk_right) and read the
    // pk_nr slab rows from pk_nl on (tmA_heads_right: box of pk_nr = pk_right + n_shift - 1 rounded up to 8 rows).
    // pk_k (pk_nl + pk_nr) <= 128.  pk_nl = 0: not packed.
    const CUtensorMap* tmA_heads_left;
    const CUtensorMap* tmA_heads_right;
    int pk_nl, pk_nr, pk_k, pk_left, pk_right;
    unsigned long long* stamp;     // profiling graph: [0] = min %globaltimer at CTA start, [1] = max at CTA end; else null
    // EPI_FINAL: this layer (ConvTranspose1d -> 32 channels, tanh) and the network's last layer
    // (ConvTranspose1d 32 -> 1, k = 7, stride 2, pad 3, output_padding 1, linear) in one kernel.  The
    // epilogue writes each activated accumulator row (positions 2m, 2m+1 x 32 channels = one 128-byte
    // row) to a shared-memory tile in the swizzled K-major layout, and a SECOND chain of tcgen05.mma
    // (M 128, N 16, K 3 x 64: rows m-1, m, m+1) turns it into the 4 predictions y[4m .. 4m+3].
    // EPI_CHAIN: the first two encoder layers (Conv1d 21 -> 32 and 32 -> 64, k 7, stride 2, tanh) in one kernel.  Two
    // consecutive tiles of this layer (2 x 128 positions x 32 channels) ARE one A tile of the next layer (128 position
    // pairs x 64): the epilogue writes them, activated, into shared memory in the swizzled K-major layout, a second
    // chain of tcgen05.mma (M 128, N 64, K 4 x 64: pair rows l-2 .. l+1) produces 125 rows of the next layer (super-tiles
    // overlap by three pair rows), and a second epilogue stores those.  This layer's activation never exists in memory.
    // tmF: the next layer's B operand, box (64, 64, 1); tmOut: ITS output, box (32, 32, 1); bias2 [n_det][64]; out2 / M2:
    // its output tensor [batch][M2][64] and rows per batch item; chain_k2: bit sh = K steps 0, 1 of shift sh hold no weight.
    const float* bias2;
    void* out2;
    int M2, chain_k2;
    CUtensorMap tmF;               // last layer as a B operand: 3-D (K = 3 x 64, N = 16, n_det), box (64, 16, 1)
    const float* fin_b;            // [n_det]
    float* pred;                   // [batch][4 M] fp32
    const float* bias;             // [n_det][N]
    void* out;                     // EPI_STORE: [batch][M][N]; EPI_POOL: [batch][M/2][N/2], 16-bit
    // EPI_POOL_HEAD: global average pool over the M/2 pooled rows, dense head, sigmoid
    const float *hw1, *hb1, *hw2, *hb2;   // [hidden][N/2], [hidden], [hidden], [1]
    int head_hidden;
    float* scores;                 // [batch]
    float* pooled_dbg;             // optional [batch][M/2][N/2] fp32 (SIMT path scratch)
#ifdef GW_TRACE
    long long* trace;              // [grid][16] cycle counters of the roles (diagnostic builds only)
#endif
    // Structural zeros of the resident-weight path, one bit per (cb, shift) at position cb * kMaxShift + shift:
    // mask_k2: K steps 0 and 1 of the segment hold no weight (a stride-2 Conv1d's outermost shift reaches one
    //          position parity only) -> two MMAs instead of four;
    // mask_nu: only the UPPER half of N holds weights (a ConvTranspose1d's outermost shift feeds odd outputs only)
    //          -> MMAs of N/2 into the upper half of the accumulator, and the block is stored at half size.
    // Skipped products are exact zeros: results do not change.  b_res_bytes = size of the resident weight image.
    unsigned long long mask_k2, mask_nu;
    int b_res_bytes;
    CUtensorMap tmBh;              // the upper-half weight blocks: box (64, N/2, 1)
    int8_t seg_of[kMaxCb][kMaxShift];     // B K-block of segment (cb, shift), -1 if the segment is empty
    int8_t seg_shift[kMaxSeg];     // per segment s: row shift, first column (SIMT kernel)
    int16_t seg_col[kMaxSeg];
};

struct GemmLaunch {
    ConvGemmParams p;
    int batch;                     // n_items * n_det
    int smem_bytes;
    int grid;                      // persistent CTAs (multiple of n_det)
    int pdl;                       // launch with programmatic stream serialization (gw_options.pdl)
};

// Virtual tile -> tile index of the layer (see ConvGemmParams::v_tiles).
__host__ __device__ __forceinline__ int map_tile(const ConvGemmParams& p, int vt) {
    return vt < p.v_left ? vt : vt + (p.tiles_m - p.v_tiles);
}

cudaError_t launch_conv_gemm_umma(const GemmLaunch& g, cudaStream_t st);
cudaError_t launch_conv_gemm_simt(const GemmLaunch& g, cudaStream_t st);
// Chooses resident/streaming B, ring depths and the shared-memory size for a layer; false if it cannot fit.
bool conv_gemm_plan(GemmLaunch& g, int sm_count);
cudaError_t probe_mufu_rate(int mode, int threads, float* results_per_clock_per_sm);   // diagnostic: activation results per clock per SM
cudaError_t probe_mma_cycles(int N, float* issue, float* complete);   // diagnostic: cycles per tcgen05.mma, N in {16..256}
cudaError_t conv_gemm_prepare();   // opt-in shared-memory attribute

// ---- bandwidth / CUDA-core kernels (gw_kernels.cu) -------------------------------------------
// Every launcher takes `stamp` (null outside the profiling graph): two 64-bit slots the kernel fills with the
// %globaltimer of its first CTA start / last CTA end, and returns the launch status.
typedef unsigned long long* Stamp;
cudaError_t launch_append(float* ring, const float* new_samples, long long* count, unsigned* ticket, int n_rows,
                          int W, int S, Stamp stamp, cudaStream_t st);
bool is_append_kernel(const void* func);   // identifies the a1 node of a captured graph
bool is_ring16_append_kernel(const void* func);
bool is_snapshot_append_kernel(const void* func);   // the fused a1 + a2 kernel (src is argument 1)
bool is_aggregate_kernel(const void* func);         // the a5 node (AggParams is argument 0)
cudaError_t launch_snapshot_append(float* ring, const float* new_samples, void* ring16, long long* count, unsigned* ticket,
                                   const int* rows_map, const float* pre, int n_streams, int channels, int n_det, int n_wit,
                                   int W, int S, int cpad, int fmt, Stamp stamp, cudaStream_t st);
cudaError_t launch_snapshot(const float* ring, float* out, const long long* count, int n_rows, int W, cudaStream_t st);
cudaError_t launch_ring16_append(const float* new_samples, void* ring16, const long long* count, const int* rows_map,
                                 int n_streams, int channels, int n_det, int n_wit, int W, int S, int cpad, int fmt,
                                 const float* pre, Stamp stamp, cudaStream_t st);
cudaError_t launch_gather(const float* ring, void* xw, const long long* count, const int* rows_map, int n_streams,
                          int channels, int n_det, int n_wit, int W, int cpad, int fmt, const float* pre, Stamp stamp,
                          cudaStream_t st, long long seg_T = 0, int seg_S = 0);
cudaError_t launch_ola_offline(const float* pred, const float* seg, const int* strain_rows, const float* hann,
                               const double* cum, float* cleaned, float* nhat_out, int B, int n_det, int W, int S,
                               long long T, const float* post, cudaStream_t st);
cudaError_t launch_final_convt(const void* x, const float* wt, const float* bias, float* pred, int batch, int n_det,
                               int L, int cpad, int K, int pad, int fmt, Stamp stamp, cudaStream_t st);
struct AggParams {
    const float* pred;         // [n][D][W] (pred_ring: ring over absolute index mod W, like acc)
    float* acc;                // [n][D][W] ring over absolute index mod W
    const float* ring;         // snapshot ring [n][C][W]
    const long long* count;
    const int* strain_rows;    // [D]
    const float* hann;         // [W]
    const float* inv_wsum;     // [W]  1 / sum of the Hann weights covering window position n
    const float* post;         // [D][2] post-processing of the estimate: (std, mean) of the strain (identity: 1, 0)
    float* final_out;          // [n][D][S] or null
    float* running_out;        // [n][D][W] or null
    float* nhat_out;           // [n][D][W] or null (test hook)
    float* clf_in;             // [n][D][Lb] or null
    int n_streams, n_det, channels, W, S, Lb, delta, agg;
    int pred_ring;
    int trigger;               // 1: let the next kernel of the stream (launched as a programmatic dependent) start early
    Stamp stamp;
    // D11: causal FIR over the stream of emitted (final) estimate samples.  fir: [fir_n] taps or null; hist: [2][n*D][kMaxFir-1]
    // the last fir_n - 1 emitted samples of the previous update (double-buffered by update parity).
    const float* fir;
    float* hist;
    int fir_n;
};
constexpr int kMaxFir = 64;        // taps of the post-filter (D11) and of the whitening filter (D12)
cudaError_t launch_aggregate(const AggParams& a, int pdl, cudaStream_t st);
cudaError_t launch_bbh_conv1(const float* x, const float* w, const float* b, void* out, int batch, int n_det, int L,
                             int cout, int cpad, int K, int pad_l, int pool, int fmt, const float* whiten, int whiten_n,
                             int pdl, Stamp stamp, cudaStream_t st);

// The whole classifier (three conv blocks + pooling + dense head) as ONE kernel, one CTA per window, every activation in
// shared memory (gw_bbh_fused.cu).  The weight images are built on the host in the exact shared-memory byte layout of the
// UMMA operands (K-major, SWIZZLE_128B) so that plain bulk copies load them:
//   w1img  [128 rows n = phase*32 + cout][64 k = (cin*2 + part)*16 + i]   block 1 as a Toeplitz matrix over 11 input samples
//   w2img  [4 tap pairs][64 rows cout][64 k = (tap & 1)*32 + cin]
//   w3img  [8 taps][128 rows cout][64 k = cin]
struct BbhFusedParams {
    const float* x;                // [batch][cin][L] fp32
    const uint8_t *w1img, *w2img, *w3img;
    const float *b1, *b2, *b3;     // [32], [64], [128] fp32 (channels past cout: 0)
    const float *hw1, *hb1, *hw2, *hb2;   // dense head: [hidden][128], [hidden], [hidden], [1]
    const float* whiten;           // D12: [cin][whiten_n] or null
    int whiten_n;
    float* scores;                 // [batch]
    int L, cin, hidden;
    Stamp stamp;
};
constexpr int kBbhW1Bytes = 128 * 128, kBbhW2Bytes = 4 * 64 * 128, kBbhW3Bytes = 8 * 128 * 128;
bool bbh_fused_supported(int L, int cin, int hidden);
cudaError_t bbh_fused_prepare();
cudaError_t launch_bbh_fused(const BbhFusedParams& p, int batch, int fmt, int pdl, cudaStream_t st);

cudaError_t launch_stamp_init(unsigned long long* stamps, int n, cudaStream_t st);   // begin slots = max, end slots = 0
int report_error(int code, const char* msg);   // records `msg` as the calling thread's gw_last_error (gw_engine.cu), returns `code`
void count_launch();               // one more kernel launched (or captured) by this library: atomic process-wide counter
long long kernel_launches();
void uncount_launches(long long n);   // captured, not launched

// Profiling stamps: %globaltimer (ns).  Thread 0 of every CTA; the end stamp follows a block-wide barrier.
__device__ __forceinline__ unsigned long long gw_globaltimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Slots per kernel: [0] min begin (ns) over CTAs, [1] max end (ns) over CTAs, and for CTA 0 alone its own begin / end in
// SM cycles ([2], [3]: clock64) and in ns ([4], [5]): cycles / ns = the SM clock that kernel actually ran at.
constexpr int kStampSlots = 6;
__device__ __forceinline__ void stamp_begin(unsigned long long* s) {
    if (s != nullptr && threadIdx.x == 0) {
        const unsigned long long t = gw_globaltimer();
        atomicMin(s, t);
        if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) { s[2] = static_cast<unsigned long long>(clock64()); s[4] = t; }
    }
}
__device__ __forceinline__ void stamp_end(unsigned long long* s) {   // call after a __syncthreads() of the whole CTA
    if (s != nullptr && threadIdx.x == 0) {
        const unsigned long long t = gw_globaltimer();
        atomicMax(s + 1, t);
        if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) { s[3] = static_cast<unsigned long long>(clock64()); s[5] = t; }
    }
}

}  // namespace gw
