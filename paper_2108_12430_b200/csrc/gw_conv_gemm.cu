// gw_conv_gemm.cu -- every Conv1d / ConvTranspose1d layer with enough channels as an implicit GEMM on
// the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM, operands staged by TMA).
//
//   D[m][n] = sum over segments (cb, a):  A[m + a][64 cb .. 64 cb + 64) . B[n][64 s .. 64 s + 64)
//
// A is a 2-D view of the channels-last input activation of one (stream, detector):
//   stride-2 Conv1d (encoder):   rows = L/2 position pairs, cols = 2 Cin (even | odd position)
//   stride-2 ConvTranspose1d:    rows = L positions,        cols = Cin; N = (even | odd output) x Cout
//   stride-1 Conv1d + pool 4:    rows = L/2 position pairs, cols = 2 Cin; N = (even | odd output) x Cout
// so every filter tap is a ROW-SHIFTED rectangular tile of the same matrix.  One output tile of 128 rows
// therefore needs a slab of 128 + (shifts - 1) input rows per 64-column block; the slab is fetched ONCE by
// one TMA box load (the layer's zero padding is TMA's out-of-bounds fill; the batch index is the third
// tensor dimension, so a slab never bleeds into the neighbouring window) and every tap's MMA reads it
// through a shared-memory descriptor whose start address is advanced by whole 128-byte rows.
//
// k_conv_gemm_umma is persistent and warp-specialised (352 threads, one CTA per SM):
//   warp 0     TMA producer: A slabs (ring of sa_stages), B K-blocks (resident once, or a ring of sb_stages)
//   warp 1     MMA issuer (one elected lane, predicated issue on the uniform datapath): tcgen05.mma into one of
//              TWO TMEM accumulator stages; in EPI_FINAL also the second chain (the network's last layer)
//   warp 10    second MMA issuer for stages that hold several tiles (odd tiles; its own A-slab sub-ring)
//   warps 2-9  epilogue: TMEM -> registers -> bias / activation / pool / head -> swizzled shared-memory staging ->
//              TMA store, overlapping the next stage's MMAs
// CTA c serves detector c % n_det (each detector has its own weights) and walks that detector's tiles
// with stride gridDim.x / n_det.  k_conv_gemm_2sm (further down) is the CTA-pair variant for N = 256.
// Two epilogues chain a SECOND layer onto the first through shared memory and a second run of tcgen05.mma: EPI_FINAL
// (the network's last two layers: the 1-channel ConvTranspose1d rides on the 32-channel one) and EPI_CHAIN (its first
// two: two tiles of layer 0 are one operand tile of layer 1); neither intermediate activation is ever stored.
// Kernels of a step are chained with programmatic dependent launch (griddepcontrol).
#include <stdio.h>

#include "gw_common.cuh"
#include "gw_ptx.cuh"

namespace gw {

// Diagnostic builds (GW_TRACE=1 python -m paper_2108_12430_b200.build): per-role cycle counters of where each
// CTA waits, written to p.trace and printed by gw_step_profile.  Compiled out of the product build.
#ifdef GW_TRACE
#define TR_DECL long long tr_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; const long long tr_t0 = clock64();
#define TR_WAIT(slot, stmt) { const long long t_ = clock64(); stmt; tr_[slot] += clock64() - t_; }
#define TR_FLUSH(base, n) if (lane == 0 && p.trace) { for (int i_ = 0; i_ < n; ++i_) p.trace[blockIdx.x * 16 + base + i_] = tr_[i_]; p.trace[blockIdx.x * 16 + base + n] = clock64() - tr_t0; }
#else
#define TR_DECL
#define TR_WAIT(slot, stmt) stmt;
#define TR_FLUSH(base, n)
#endif

constexpr int kEpiWarps = 8;
constexpr int kGemmThreads = 64 + kEpiWarps * 32 + 32;   // producer warp, MMA warp, 8 epilogue warps, second MMA warp
constexpr int kMmaWarp2 = 2 + kEpiWarps;                  // warp index of the second MMA issuer
constexpr int kAccCols = 256;                        // TMEM columns of one accumulator stage
constexpr int kSmemBudget = 225 * 1024;
constexpr int kFixedSmem = 1024 /*alignment slack*/ + 1024 /*bias*/ + 1024 /*barriers, tmem slot*/;
constexpr int kFinBlock = 16 * 128;                  // EPI_FINAL: one K block (64) of the last layer's B operand, N = 16 rows
constexpr int kFinalScratch = 3 * kFinBlock;         // EPI_FINAL: last-layer B operand, 3 row shifts
constexpr int kFinTile = kTileM * 128;               // EPI_FINAL: one activated tile, 128 rows x 128 bytes
constexpr int kFinN = 16;                            // EPI_FINAL: N of the second MMA chain (4 real columns)
constexpr int kFinCol = 128;                         // EPI_FINAL: TMEM column of the second chain's accumulators in a stage
constexpr int kOutStage = kEpiWarps * 4096;          // output staging: 32 rows x 128 bytes per epilogue warp
constexpr int kChainRows = 125;                      // EPI_CHAIN: rows of the second layer one super-tile produces
constexpr int kChainTile = kTileM * 128;             // EPI_CHAIN: the second layer's A tile (two activated tiles of this layer)
constexpr int kChainStg = 4 * kChainTile + 1024;     // EPI_CHAIN: offset of the second epilogue's staging (2 x 2 KiB per warp) behind
                                                     // the four A tiles ([stage][super-tile of the stage]) and 1 KiB the shifted
                                                     // reads of the last rows run into
constexpr int kChainOut = kChainStg + kEpiWarps * 4096;
constexpr int kChainBlock = 64 * 128;                // EPI_CHAIN: one K block of the second layer's B operand (N = 64 rows)
constexpr int kChainScratch = 4 * kChainBlock;
// first row (position) of this layer's virtual tile vt in chain mode: super-tile s = vt / 2 covers the second layer's rows
// [125 s, 125 s + 125), which read its input pair rows 125 s - 2 .. 125 s + 125, i.e. positions from 250 s - 4 on
__host__ __device__ __forceinline__ int chain_m0(int vt) { return (vt >> 1) * (2 * kChainRows) - 4 + (vt & 1) * kTileM; }

__host__ __device__ __forceinline__ int slab_bytes_of(int slab_rows) { return (slab_rows * 128 + 1023) & ~1023; }
__host__ __device__ __forceinline__ int head_scratch_bytes(int N, int hidden) {
    return ((64 * (N / 2 + 1) + N / 2 + hidden) * 4 + 1023) & ~1023;
}

bool conv_gemm_plan(GemmLaunch& g, int sm_count) {
    ConvGemmParams& p = g.p;
    const int b_block = p.N * 128;
    const int sl = slab_bytes_of(p.slab_rows + (p.two_sm ? p.pk_nl : 0));
    if (p.two_sm) {
        // CTA-pair kernel: N = 256 store layers with an even number of tiles; half weight blocks of 16 KiB
        const int pairs = sm_count / 2;
        // ring input (incremental path): needs the per-head tensor maps; the pair works on virtual tiles 2u, 2u + 1
        bool ok = p.epi == EPI_STORE && p.N == 256 && (p.a_count == nullptr || p.tmA_heads != nullptr) &&
                  (p.pk_nl ? (g.batch / p.n_det) % (2 * p.pk_k) == 0 && p.tmA_heads_left != nullptr && p.tmA_heads_right != nullptr
                           : p.v_tiles % 2 == 0) && pairs >= p.n_det;
        for (int ob = 2; ok && ob >= 1; --ob) {
            const int fixed = kFixedSmem + ob * kOutStage;
            const int sa = p.n_cb < 2 ? 2 : (p.n_cb > 8 ? 8 : p.n_cb);
            int sb = (kSmemBudget - fixed - sa * sl) / (128 * 128);
            if (sb > 8) sb = 8;
            if (sb < 3) continue;
            p.out_bufs = ob; p.b_resident = 0; p.sa_stages = sa; p.sb_stages = sb;
            g.smem_bytes = fixed + sb * 128 * 128 + sa * sl;
            g.grid = 2 * (pairs - pairs % p.n_det);
            return true;
        }
        p.two_sm = 0;
        p.pk_nl = 0;                                   // packing exists in the pair kernel only
    }
    // EPI_STORE stages its output through shared memory for TMA stores: one 4 KiB buffer per epilogue warp,
    // two when the operands leave room (thin layers)
    p.out_bufs = 0;
    if (p.epi == EPI_FINAL) p.out_bufs = 2;               // four activated tiles: [accumulator stage][tile in stage]
    if (p.epi == EPI_STORE) {
        int nh = 0;
        for (unsigned long long m = p.mask_nu; m; m &= m - 1) ++nh;
        const int rb = p.n_seg * b_block - nh * (b_block / 2);
        const int b_need = rb <= 132 * 1024 ? rb : 4 * b_block;
        p.out_bufs = (kFixedSmem + 2 * kOutStage + b_need + 4 * sl <= kSmemBudget) ? 2 : 1;
    }
    const int fixed = kFixedSmem + (p.epi == EPI_POOL_HEAD ? head_scratch_bytes(p.N, p.head_hidden) : 0) +
                      (p.epi == EPI_FINAL ? kFinalScratch : 0) + (p.epi == EPI_CHAIN ? kChainScratch + kChainOut : 0) +
                      p.out_bufs * kOutStage;
    int b_bytes;
    int n_half = 0;
    for (unsigned long long m = p.mask_nu; m; m &= m - 1) ++n_half;
    const int res_bytes = p.n_seg * b_block - n_half * (b_block / 2);      // upper-half-only blocks are stored at half size
    if (res_bytes <= 132 * 1024 && fixed + res_bytes + 2 * sl <= kSmemBudget) {
        p.b_resident = 1; p.sb_stages = 0; b_bytes = res_bytes; p.b_res_bytes = res_bytes;
    } else {
        p.mask_k2 = 0; p.mask_nu = 0;                                      // streamed weights: every block in full
        p.b_resident = 0;
        p.sb_stages = p.n_seg < 4 ? p.n_seg : 4;
        while (p.sb_stages > 1 && fixed + p.sb_stages * b_block + 2 * sl > kSmemBudget) p.sb_stages--;
        b_bytes = p.sb_stages * b_block;
    }
    int sa = (kSmemBudget - fixed - b_bytes) / sl;
    if (sa < 2) return false;
    if (sa > 8) sa = 8;
    p.sa_stages = sa;
    g.smem_bytes = fixed + b_bytes + sa * sl;
    g.grid = sm_count - sm_count % p.n_det;
    // tiles per stage: when the whole launch is less than one wave of full stages (few streams: the latency
    // regime), smaller units spread it over more CTAs -- the smallest unit count that still fits one wave wins.
    // With more work than that the full stage stays (measured at n = 16: smaller units did not pay).
    p.g_tiles = 0;
    if (p.epi == EPI_STORE && g.batch > 0) {
        const int n_items = g.batch / p.n_det, workers = g.grid / p.n_det;
        for (int G = kAccCols / p.N; G >= 2; G /= 2) {
            const long long units = static_cast<long long>(n_items) * ((p.v_tiles + G - 1) / G);
            if (units > workers) break;
            p.g_tiles = G;
        }
    }
    return true;
}

template <int FMT>
__device__ __forceinline__ uint32_t pack_pair_t(float a, float b) {
    if (FMT == FMT_BF16) {
        __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
        return *reinterpret_cast<uint32_t*>(&v);
    }
    __half2 v = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// Activation + rounding to the storage type of two neighbouring outputs.
// tanh on the MUFU pipe is what bounds the thin layers' epilogue (16 lanes per clock per SM): the exact
// form 1 - 2/(1 + e^{2v}) costs two MUFU ops (ex2, rcp) and six FP32 ops per element, tanh.approx.f32 one
// MUFU op (relative error 2^-11: about one fp16 rounding step; SURVEY.md A18 allows it and the parity
// tests hold the result to north_star's tolerances).  fp16 takes the one-op form, bf16 the exact one.  tanh.approx.f16x2 was
// tried: ptxas splits it into two MUFU.TANH.F16, so it saves nothing and is less accurate.
#ifdef GW_BF16_APPROX_TANH
constexpr bool kBf16ExactTanh = false;
#else
constexpr bool kBf16ExactTanh = true;
#endif
template <int ACT, int FMT>
__device__ __forceinline__ uint32_t act_pack_t(float a, float b) {
    if (ACT == ACT_TANH) {
        if (FMT == FMT_BF16 && kBf16ExactTanh) {
            // bf16 keeps the exact form: its per-element error budget is already spent on storage rounding
            // and every flipped rounding costs 2^-8
            const float ea = __expf(2.f * a), eb = __expf(2.f * b);
            return pack_pair_t<FMT>(1.f - __fdividef(2.f, 1.f + ea), 1.f - __fdividef(2.f, 1.f + eb));
        }
        float ta, tb;
        asm("tanh.approx.f32 %0, %1;" : "=f"(ta) : "f"(a));
        asm("tanh.approx.f32 %0, %1;" : "=f"(tb) : "f"(b));
        return pack_pair_t<FMT>(ta, tb);
    }
    if (ACT == ACT_RELU) return pack_pair_t<FMT>(fmaxf(a, 0.f), fmaxf(b, 0.f));
    return pack_pair_t<FMT>(a, b);
}

// The same activation on one value, kept in fp32 (EPI_FINAL feeds it straight into the last layer).
template <int ACT, int FMT>
__device__ __forceinline__ float act_f32_t(float a) {
    if (ACT == ACT_TANH) {
        if (FMT == FMT_BF16 && kBf16ExactTanh) return 1.f - __fdividef(2.f, 1.f + __expf(2.f * a));
        float t;
        asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(a));
        return t;
    }
    if (ACT == ACT_RELU) return fmaxf(a, 0.f);
    return a;
}

__device__ __forceinline__ float act_apply(float v, int act) {
    if (act == ACT_TANH) {
        // tanh(v) = 1 - 2/(1 + e^{2v}): two MUFU ops (ex2, rcp), absolute error ~1e-7.  The one-op
        // tanh.approx.f32 (relative error 2^-11) is as large as a bf16 rounding step and 4x an fp16 one,
        // and it flips ~10% of the storage roundings.
        const float e = __expf(2.f * v);
        return 1.f - __fdividef(2.f, 1.f + e);
    }
    if (act == ACT_RELU) return fmaxf(v, 0.f);
    return v;
}

__device__ __forceinline__ uint32_t pack_pair(float a, float b, int fmt) {
    if (fmt == FMT_BF16) {
        __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
        return *reinterpret_cast<uint32_t*>(&v);
    }
    __half2 v = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// Row-shifted operand views: a descriptor whose start address is advanced by whole 128-byte rows inside
// a 1024-byte aligned SWIZZLE_128B slab needs NO base-offset (bits 49-51 stay 0): the tensor core
// derives the swizzle phase from the absolute shared-memory address bits, exactly as TMA did when it
// wrote the slab.  Measured on B200: base_offset = 0 matches the oracle, base_offset = (addr >> 7) & 7
// gives garbage (round-1 bring-up measurement).

// EPI / ACT / FMT are compile-time so that the per-element epilogue loop is straight-line code the
// compiler can unroll and interleave (with run-time branches inside it, each element's MUFU latency
// chain was exposed: ~120 cycles per element with only four epilogue warps to hide it).
//
// One accumulator stage is kAccCols = 256 TMEM columns and holds G = 256 / N consecutive output tiles
// (EPI_STORE; G = 1 for the pooled epilogues), so that thin layers (N = 32, 64) hand over 8 or 4 tiles
// per mbarrier round trip instead of one.  Two stages (512 columns) double-buffer MMA against epilogue.
// ZONE: the incremental path's output forms (mirror-ring stores, prediction ring, dead-quadrant skipping) exist in their
// own instantiation, so that the whole-window kernels of the full step carry none of it.
// NT: GEMM N as a compile-time constant (0: read from the parameters) -- the whole-window DeepClean layers get their own
// instantiation per width, so that the instruction descriptor, the weight-block stride and the epilogue's chunk -> tile
// map are constants.
template <int EPI, int ACT, int FMT, bool ZONE, int NT>
__global__ void __launch_bounds__(kGemmThreads, 1) k_conv_gemm_umma(const __grid_constant__ ConvGemmParams p,
                                                                    int n_items) {
    const int pN = NT ? NT : p.N;
    const int out_ring_div = ZONE ? p.out_ring_div : 0, pred_ring = ZONE ? p.pred_ring : 0;
    const int z_left = ZONE ? p.z_left : 0, z_right = ZONE ? p.z_right : 0;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int b_block = pN * 128;
    const int sl = slab_bytes_of(p.slab_rows);
    const int sa = p.sa_stages, sb = p.sb_stages;
    uint8_t* smem_out = smem;                                                // [out_bufs][8 warps][4 KiB]
    uint8_t* smem_b = smem + (EPI == EPI_CHAIN ? kChainOut : p.out_bufs * kOutStage);
    uint8_t* smem_a = smem_b + (p.b_resident ? p.b_res_bytes : sb * b_block);
    uint8_t* after_a = smem_a + sa * sl;
    float* bias_s = reinterpret_cast<float*>(after_a);                       // [N]
    uint64_t* bars = reinterpret_cast<uint64_t*>(after_a + 1024);
    uint64_t* a_full = bars;                 // [sa]
    uint64_t* a_empty = a_full + 8;          // [sa]
    uint64_t* b_full = a_empty + 8;          // [sb]
    uint64_t* b_empty = b_full + 4;          // [sb]
    uint64_t* bres_bar = b_empty + 4;        // [1]
    uint64_t* tmem_full = bres_bar + 1;      // [2]
    uint64_t* tmem_empty = tmem_full + 2;    // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_empty + 2);
    uint64_t* stg_full = bars + 32;          // [2 stages][2 tiles] EPI_FINAL: activated tile written to shared memory
    uint64_t* fin_full = stg_full + 4;       // [2][2]              EPI_FINAL: second MMA chain of that tile complete
    float* head_s = reinterpret_cast<float*>(after_a + 2048);                // EPI_POOL_HEAD scratch
    uint8_t* smem_fin = after_a + 2048;                                      // EPI_FINAL: last layer's B operand (1024-aligned)

    stamp_begin(p.stamp);
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x / 32, 0);   // provably warp-uniform: role branches and
                                                                      // everything under them use the uniform datapath
    const int lane = threadIdx.x % 32;
    const int det = blockIdx.x % p.n_det;
    const int worker = blockIdx.x / p.n_det;
    const int n_workers = gridDim.x / p.n_det;
    const int G = EPI == EPI_STORE ? (p.g_tiles ? p.g_tiles : kAccCols / pN) : EPI == EPI_CHAIN ? 4 : EPI == EPI_FINAL ? 2 : 1;   // tiles per accumulator stage
    const int spi = (p.v_tiles + G - 1) / G;                                 // super-tiles per batch item (virtual tiles:
                                                                             // all of them, or the two recomputed zones)
    // Two MMA-issuing warps share a stage when it holds several tiles (even tiles: warp 1, odd tiles: warp
    // kMmaWarp2).  Below N = 128 an MMA is bound by its shared-memory operand read (32 + N/4 cycles, measured:
    // profiles/r01_mma_rate_microbench.txt) and a single issuing warp ADDS ~30 cycles of descriptor arithmetic per
    // instruction (GW_TRACE: 69 / 76 / 87 cycles per MMA at N = 32 / 64 / 128); two warps hide one behind the other.
    // Each MMA warp owns its own sub-ring of A-slab stages (even tiles: stages [0, ring0), odd tiles: the rest): a
    // stage whose fills alternate between two waiters could be one mbarrier phase ahead of one of them, and a
    // parity wait cannot tell (TMA completions are unordered).
    const int n_mma = (G >= 2 && p.b_resident && sa >= 4) ? 2 : 1;
    const int ring0 = n_mma == 2 ? (sa + 1) / 2 : sa;                       // stages of sub-ring 0
    const int total = n_items * spi;

    if (warp == 0) {
        if (lane == 0) {
            tma_prefetch_desc(&p.tmA);
            tma_prefetch_desc(&p.tmB);
            if (EPI == EPI_FINAL || EPI == EPI_CHAIN) tma_prefetch_desc(&p.tmF);
            for (int i = 0; i < sa; ++i) { mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1); }
            for (int i = 0; i < sb; ++i) { mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1); }
            mbar_init(bres_bar, 1);
            for (int i = 0; i < 2; ++i) { mbar_init(&tmem_full[i], n_mma); mbar_init(&tmem_empty[i], kEpiWarps); }
            for (int i = 0; i < 4; ++i) { mbar_init(&stg_full[i], EPI == EPI_CHAIN ? kEpiWarps : 4); mbar_init(&fin_full[i], 1); }
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc(tmem_slot, 2 * kAccCols);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);   // uniform register
    // Programmatic dependent launch: the next kernel of the step may be scheduled onto SMs as this grid's
    // CTAs retire (its prologue and weight loads overlap our tail); we ourselves touch nothing the previous
    // kernel wrote before griddep_wait().  Weights and biases are constants of the engine.
    griddep_launch_dependents();

    if (warp == 0) {
        // ------------------------------------------------------------------------ TMA producer
        if (lane == 0) {
            if (p.b_resident) {
                mbar_arrive_expect_tx(bres_bar, p.b_res_bytes + (EPI == EPI_FINAL ? kFinalScratch : 0) + (EPI == EPI_CHAIN ? kChainScratch : 0));
                int off = 0;                                   // blocks in issue order (cb outer, shift inner)
                for (int cb = 0; cb < p.n_cb; ++cb)
                    for (int sh = 0; sh < p.n_shift; ++sh) {
                        const int s = p.seg_of[cb][sh];
                        if (s < 0) continue;
                        if ((p.mask_nu >> (cb * kMaxShift + sh)) & 1ull) {
                            tma_load_3d(smem_b + off, &p.tmBh, bres_bar, s * kSegK, pN / 2, det);
                            off += b_block / 2;
                        } else {
                            tma_load_3d(smem_b + off, &p.tmB, bres_bar, s * kSegK, 0, det);
                            off += b_block;
                        }
                    }
                if (EPI == EPI_FINAL)
                    for (int s = 0; s < 3; ++s) tma_load_3d(smem_fin + s * kFinBlock, &p.tmF, bres_bar, s * kSegK, 0, det);
                if (EPI == EPI_CHAIN)
                    for (int s = 0; s < 4; ++s) tma_load_3d(smem_fin + s * kChainBlock, &p.tmF, bres_bar, s * kSegK, 0, det);
            }
            griddep_wait();
            int ib = 0;
            int rs0 = 0, rs1 = 0; uint32_t rp0 = 0, rp1 = 0;                 // position and phase in each sub-ring
            TR_DECL
            // mirror-ring source: the window starts at ring row (count mod W) / div (see ConvGemmParams); with a tensor map
            // per window head the map itself is based there (and rows outside the window are zero fill)
            const int ring_h0 = p.a_count ? static_cast<int>(*p.a_count % p.a_ring_W) : 0;
            const CUtensorMap* tmA = p.tmA_heads ? p.tmA_heads + ring_h0 / p.head_div : &p.tmA;
            const int row_off = (p.a_count && !p.tmA_heads) ? ring_h0 / p.a_ring_div : 0;
            for (int w = worker; w < total; w += n_workers) {
                const int u = p.reverse ? total - 1 - w : w;
                const int batch = (u / spi) * p.n_det + det;
                for (int g = 0; g < G; ++g) {
                    const int vt = (u % spi) * G + g;
                    if (vt >= p.v_tiles) break;
                    const int m0 = EPI == EPI_CHAIN ? chain_m0(vt) : map_tile(p, vt) * p.tile_stride + p.tile_row0;
                    for (int cb = 0; cb < p.n_cb; ++cb) {
                        const bool second = n_mma == 2 && (g & 1);
                        const int stage = second ? ring0 + rs1 : rs0;
                        TR_WAIT(0, mbar_wait(&a_empty[stage], (second ? rp1 : rp0) ^ 1))
                        mbar_arrive_expect_tx(&a_full[stage], p.slab_rows * 128);
                        if (p.a_4d) tma_load_4d(smem_a + stage * sl, &p.tmA, &a_full[stage], cb * kSegK, m0 + p.a_min, det, u / spi);
                        else tma_load_3d(smem_a + stage * sl, tmA, &a_full[stage], cb * kSegK, m0 + p.a_min + row_off, batch);
                        if (second) { if (++rs1 == sa - ring0) { rs1 = 0; rp1 ^= 1; } }
                        else if (++rs0 == ring0) { rs0 = 0; rp0 ^= 1; }
                        if (!p.b_resident) {
                            for (int sh = 0; sh < p.n_shift; ++sh) {
                                const int s = p.seg_of[cb][sh];
                                if (s < 0) continue;
                                const int bs = ib % sb;
                                TR_WAIT(1, mbar_wait(&b_empty[bs], ((ib / sb) & 1) ^ 1))
                                mbar_arrive_expect_tx(&b_full[bs], b_block);
                                tma_load_3d(smem_b + bs * b_block, &p.tmB, &b_full[bs], s * kSegK, 0, det);
                                ++ib;
                            }
                        }
                    }
                }
            }
            TR_FLUSH(0, 2)
        }
    } else if (warp == 1 || (warp == kMmaWarp2 && n_mma == 2)) {
        // -------------------------------------------------------------------------- MMA issuer
        const int mw = warp == 1 ? 0 : 1;
        // The whole warp walks the loops; one elected lane issues the MMAs and commits, selected by an
        // instruction PREDICATE on the tcgen05 instruction itself (umma_f16_if), never by a branch: inside a
        // divergent `if (elect)` block the compiler computes every descriptor in vector registers and moves
        // it to uniform registers one R2UR at a time; clock64 stamps put that block at ~330 cycles fixed
        // plus ~40 per MMA, which bounded every layer with N <= 128 (an MMA there executes in 16..64 cycles).
        // Which shifts exist for column block cb is a 6-bit field of the register `shmask`.
        const uint32_t idesc = umma_idesc_f16(FMT, kTileM, pN);
        if (p.b_resident) mbar_wait(bres_bar, 0);
        const uint32_t smem_a_u32 = smem_u32(smem_a), smem_b_u32 = smem_u32(smem_b);
        const bool resident = p.b_resident != 0;
        const bool ring = p.a_count != nullptr && p.tmA_heads == nullptr;   // window-edge rows must be cleared by hand
        const int n_cb = p.n_cb, n_shift = p.n_shift;
        const uint32_t b_step = static_cast<uint32_t>(b_block) >> 4;       // descriptor units per B K-block
        const uint32_t idesc_half = umma_idesc_f16(FMT, kTileM, pN / 2);
        const unsigned long long mask_k2 = p.mask_k2, mask_nu = p.mask_nu;
        unsigned long long shmask = 0;
        for (int cb = 0; cb < n_cb; ++cb)
            for (int sh = 0; sh < n_shift; ++sh)
                if (p.seg_of[cb][sh] >= 0) shmask |= 1ull << (cb * kMaxShift + sh);
        const uint32_t leader = elect_one() ? 1u : 0u;  // the one lane that issues (same lane every time)
        int it = 0;
        TR_DECL
        const int ring_base = mw ? ring0 : 0, ring_size = mw ? sa - ring0 : ring0;
        int stage = 0; uint32_t a_phase = 0;            // position in this warp's A sub-ring
        int bs = 0; uint32_t b_phase = 0;               // B ring position (streaming mode)
        // EPI_FINAL: the second chain of super-tile `itp` (both tiles): D row i = rows i, i+1, i+2 of the
        // activated tile (tile rows m-1, m, m+1 of output row m = i + 1) times the last layer's three K blocks.
        const uint32_t idesc_fin = umma_idesc_f16(FMT, kTileM, kFinN);
        const uint32_t fin_lo = umma_desc_lo(smem_u32(smem_fin));
        const uint32_t stg_lo = umma_desc_lo(smem_u32(smem_out));
        auto issue_final = [&](int itp) {
            const int accp = itp & 1;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (n_mma == 2 && h != mw) continue;
                TR_WAIT(3, mbar_wait(&stg_full[accp * 2 + h], (itp >> 1) & 1))
                tc_fence_after();
                const uint32_t d_fin = tmem_base + accp * kAccCols + kFinCol + h * kFinN;
                const uint32_t a_t = stg_lo + static_cast<uint32_t>((accp * 2 + h) * kFinTile >> 4);
                // shift 0 (row m-1) reaches the outputs only through its odd position (columns 32..63: K steps 2, 3):
                // tap j = r + 3 + 4 - 2 par is valid for par = 1 alone, so K steps 0, 1 of that block are all zero
#pragma unroll
                for (int sh = 0; sh < 3; ++sh)
#pragma unroll
                    for (int k = (sh == 0 ? 2 : 0); k < kSegK / 16; ++k)
                        umma_f16_if(leader, d_fin, umma_desc_make(a_t + 8u * sh + 2 * k),
                                    umma_desc_make(fin_lo + static_cast<uint32_t>(sh * kFinBlock >> 4) + 2 * k), idesc_fin,
                                    (sh == 0 && k == 2) ? 0u : 1u);
                umma_commit_if(leader, &fin_full[accp * 2 + h]);
            }
        };
        // EPI_CHAIN: the second layer on super-tile `itp`: D row i = pair rows i .. i + 3 of the activated A tile (input pair
        // rows l - 2 .. l + 1 of output row l = 125 s + i) times the second layer's four K blocks; the same K steps in the
        // same order as that layer's own kernel issues them (chain_k2: K steps 0, 1 of a block hold no weight).
        const uint32_t idesc_ch = umma_idesc_f16(FMT, kTileM, 64);
        auto issue_chain = [&](int itp) {
          const int accp = itp & 1;
#pragma unroll
          for (int j = 0; j < 2; ++j) {                    // the stage's two super-tiles: one per MMA warp
            if (n_mma == 2 && j != mw) continue;
            TR_WAIT(3, mbar_wait(&stg_full[accp * 2 + j], (itp >> 1) & 1))
            tc_fence_after();
            const uint32_t d_ch = tmem_base + accp * kAccCols + kFinCol + j * 64;
            const uint32_t a_t = stg_lo + static_cast<uint32_t>((accp * 2 + j) * kChainTile >> 4);
            uint32_t first = 0;
#pragma unroll
            for (int sh = 0; sh < 4; ++sh) {
                const uint32_t bl = fin_lo + static_cast<uint32_t>(sh * kChainBlock >> 4);
                if ((p.chain_k2 >> sh) & 1) {
#pragma unroll
                    for (int k = 2; k < kSegK / 16; ++k)
                        umma_f16_if(leader, d_ch, umma_desc_make(a_t + 8u * sh + 2 * k), umma_desc_make(bl + 2 * k), idesc_ch, first | (k - 2));
                } else {
#pragma unroll
                    for (int k = 0; k < kSegK / 16; ++k)
                        umma_f16_if(leader, d_ch, umma_desc_make(a_t + 8u * sh + 2 * k), umma_desc_make(bl + 2 * k), idesc_ch, first | k);
                }
                first = 1;
            }
            umma_commit_if(leader, &fin_full[accp * 2 + j]);
          }
        };
        for (int w = worker; w < total; w += n_workers, ++it) {
            const int u = p.reverse ? total - 1 - w : w;
            const int acc = it & 1;
            TR_WAIT(0, mbar_wait(&tmem_empty[acc], ((it >> 1) & 1) ^ 1))
            tc_fence_after();
            const int g_end = min(G, p.v_tiles - (u % spi) * G);
            for (int g = 0; g < g_end; ++g) {
                if (n_mma == 2 && (g & 1) != mw) continue;                 // the other warp's tile
                const uint32_t d_tmem = tmem_base + acc * kAccCols + g * pN;
                uint32_t accumulate = 0;
                uint32_t b_lo = umma_desc_lo(smem_b_u32);                  // resident: block 0 of B
                for (int cb = 0; cb < n_cb; ++cb) {
                    const uint32_t m = static_cast<uint32_t>(shmask >> (cb * kMaxShift)) & ((1u << kMaxShift) - 1);
                    const int astage = ring_base + stage;
                    TR_WAIT(1, mbar_wait(&a_full[astage], a_phase))
                    tc_fence_after();
                    if (ring) {
                        // window-edge zero padding: slab rows whose logical row is outside [0, M) hold
                        // neighbouring ring samples; clear them (whole 128-byte rows: swizzle-agnostic)
                        const int lo = (EPI == EPI_CHAIN ? chain_m0((u % spi) * G + g) : map_tile(p, (u % spi) * G + g) * p.tile_stride + p.tile_row0) + p.a_min;
                        if (lo < 0 || lo + p.slab_rows > p.a_rows) {
                            uint8_t* slab = smem_a + astage * sl;
                            for (int idx = lane; idx < p.slab_rows * 8; idx += 32) {
                                const int lr = lo + (idx >> 3);
                                if (lr < 0 || lr >= p.a_rows)
                                    *reinterpret_cast<uint4*>(slab + (idx >> 3) * 128 + (idx & 7) * 16) = make_uint4(0, 0, 0, 0);
                            }
                            fence_proxy_async();
                            __syncwarp();
                        }
                    }
                    const uint32_t a_lo = umma_desc_lo(smem_a_u32 + astage * sl);
                    if (resident) {
                        uint32_t acc_flag = accumulate, bl = b_lo;
                        const uint32_t mk2 = static_cast<uint32_t>(mask_k2 >> (cb * kMaxShift)), mnu = static_cast<uint32_t>(mask_nu >> (cb * kMaxShift));
                        for (int sh = 0; sh < n_shift; ++sh) {
                            if (!((m >> sh) & 1u)) continue;
                            const uint32_t a_lo_s = a_lo + 8u * sh;        // +128 bytes = one slab row
                            if ((mnu >> sh) & 1u) {                        // weights in the upper half of N only (half-size block)
#pragma unroll
                                for (int k = 0; k < kSegK / 16; ++k)
                                    umma_f16_if(leader, d_tmem + pN / 2, umma_desc_make(a_lo_s + 2 * k), umma_desc_make(bl + 2 * k), idesc_half, 1u);
                                bl += b_step / 2;
                            } else if ((mk2 >> sh) & 1u) {                 // K steps 0, 1 hold no weight
#pragma unroll
                                for (int k = 2; k < kSegK / 16; ++k)
                                    umma_f16_if(leader, d_tmem, umma_desc_make(a_lo_s + 2 * k), umma_desc_make(bl + 2 * k), idesc, acc_flag | (k - 2));
                                bl += b_step;
                            } else {
#pragma unroll
                                for (int k = 0; k < kSegK / 16; ++k)       // +32 bytes along K: +2 in (addr >> 4)
                                    umma_f16_if(leader, d_tmem, umma_desc_make(a_lo_s + 2 * k), umma_desc_make(bl + 2 * k), idesc, acc_flag | k);
                                bl += b_step;
                            }
                            acc_flag = 1;
                        }
                        umma_commit_if(leader, &a_empty[astage]);          // slab free once these MMAs retire
                        b_lo = bl;
                    } else {
                        for (int sh = 0; sh < n_shift; ++sh) {
                            if (!((m >> sh) & 1u)) continue;
                            TR_WAIT(2, mbar_wait(&b_full[bs], b_phase))
                            tc_fence_after();
                            const uint32_t bl = umma_desc_lo(smem_b_u32 + bs * b_block);
                            const uint32_t a_lo_s = a_lo + 8u * sh;
                            const bool last = (m >> (sh + 1)) == 0;
#pragma unroll
                            for (int k = 0; k < kSegK / 16; ++k)
                                umma_f16_if(leader, d_tmem, umma_desc_make(a_lo_s + 2 * k), umma_desc_make(bl + 2 * k), idesc, accumulate | k);
                            umma_commit_if(leader, &b_empty[bs]);
                            if (last) umma_commit_if(leader, &a_empty[astage]);
                            accumulate = 1;
                            if (++bs == sb) { bs = 0; b_phase ^= 1; }
                        }
                    }
                    accumulate = 1;
                    if (++stage == ring_size) { stage = 0; a_phase ^= 1; }
                }
            }
            umma_commit_if(leader, &tmem_full[acc]);                       // accumulator stage complete
            if (EPI == EPI_FINAL && it > 0) issue_final(it - 1);           // behind this stage's MMAs in the pipe
            if (EPI == EPI_CHAIN && it > 0) issue_chain(it - 1);
        }
        if (EPI == EPI_FINAL && it > 0) issue_final(it - 1);
        if (EPI == EPI_CHAIN && it > 0) issue_chain(it - 1);
        if (mw == 0) { TR_FLUSH(3, 4) }
    } else if (warp < kMmaWarp2) {
        // ------------------------------------------------------------- epilogue warps 2..9 (8 warps)
        const int quad = warp % 4;                             // TMEM lane quadrant this warp may read
        const int hsel = (warp - 2) / 4;                       // which half of the 32-column chunks
        const int row_in_tile = quad * 32 + lane;
        const int et = threadIdx.x - 64;                       // 0..255
        for (int i = et; i < pN; i += kEpiWarps * 32) bias_s[i] = __ldg(p.bias + static_cast<size_t>(det) * pN + i);
        if (EPI == EPI_CHAIN && et < 64) bias_s[64 + et] = __ldg(p.bias2 + static_cast<size_t>(det) * 64 + et);   // second layer's
        asm volatile("bar.sync 1, 256;" ::: "memory");
        // the four 32-column chunks this warp owns in every stage: tile-in-stage g and first column col0
        int ch_g[4], ch_col[4];
        const uint32_t bias_u32 = smem_u32(bias_s);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int c = 4 * (i / 2) + 2 * hsel + (i % 2);    // pairs of ADJACENT chunks: 128 contiguous bytes per row
            ch_g[i] = (32 * c) / pN;
            ch_col[i] = (32 * c) % pN;
        }
        griddep_wait();                                        // before the first global store of this grid
        // incremental path: window start inside the output mirror ring / the prediction ring (the append kernel of
        // this update has advanced the counter; nothing changes it while the conv kernels run)
        const int ring_h = (out_ring_div || pred_ring) ? static_cast<int>(*p.a_count % p.a_ring_W) : 0;
        const int out_off = out_ring_div ? ring_h / out_ring_div : 0;
        // One 32-row box of this tile at window row `row` (whole warp calls it; lane 0 issues the TMA stores).  Mirror
        // ring: ring row r = out_off + row, and every row is stored a second time at its twin r +- M.  A box that
        // straddles row M has twins on both sides: those of its rows below M go out with a TMA store that the tensor
        // map clips at 2M; the few rows at or above M are copied to ring rows 0.. by the lanes (TMA stores do not take
        // negative coordinates).  row_bytes = 128 (N >= 64: 128B swizzle) or 64 (N = 32: 64B swizzle).
        auto store_box = [&](uint32_t src, int col, int row, int b, int row_bytes) {
            const int r = out_off + row;
            if (lane == 0) {
                tma_store_3d(&p.tmOut, src, col, r, b);
                if (out_ring_div) {
                    if (r >= p.M) tma_store_3d(&p.tmOut, src, col, r - p.M, b);
                    else tma_store_3d(&p.tmOut, src, col, r + p.M, b);
                }
            }
            if (out_ring_div && r < p.M && r + 31 >= p.M && r + lane >= p.M) {
                uint8_t* dst = reinterpret_cast<uint8_t*>(p.out) +
                               ((static_cast<size_t>(b) * 2 * p.M + (r + lane - p.M)) * pN + col) * 2;
                const int units = row_bytes / 16;
                for (int u = 0; u < units; ++u) {
                    const int su = row_bytes == 128 ? (u ^ (lane & 7)) : (u ^ ((lane >> 1) & 3));
                    *reinterpret_cast<float4*>(dst + 16 * u) = lds_f4(src + lane * row_bytes + (su << 4));
                }
            }
        };
        // zone launches (EPI_STORE): rows [r0, r0 + 32) of the layer hold a recomputed row iff they reach into the first
        // z_left or the last z_right rows
        auto quad_live = [&](int vt) -> bool {
            if ((z_left | z_right) == 0) return true;
            const int r0 = map_tile(p, vt) * kTileM + quad * 32;
            return r0 < z_left || r0 + 32 > p.M - z_right;
        };
        auto fin_row_live = [&](int orow) -> bool {            // EPI_FINAL zone launches: is this output row recomputed?
            return (z_left | z_right) == 0 || orow < z_left || orow >= p.M - z_right;
        };
        const float fin_bias = EPI == EPI_FINAL ? __ldg(p.fin_b + det) : 0.f;
        // EPI_CHAIN, second epilogue: the 2 x 125 rows the two super-tiles `s_prev`, `s_prev + 1` of batch item `b_prev`
        // produced (their chains were issued one iteration ago and have long retired).  Warp (quad, hsel): rows [32 quad, +32),
        // channels [32 hsel, +32) of both; bias, tanh, 16-bit, through this warp's two 2 KiB staging buffers; quadrants 0-2 leave
        // with one TMA store each (32 rows x 64 bytes, clipped at the tensor's last row), quadrant 3 holds 29 live rows, which
        // its lanes copy out themselves.
        const uint32_t chain_stg = smem_u32(smem_out) + kChainStg + (warp - 2) * 4096;   // two 2 KiB boxes: one per super-tile of the stage
        auto chain_emit = [&](int accp, uint32_t parity, int b_prev, int s_prev) {
            uint32_t r[2][32];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                mbar_wait(&fin_full[accp * 2 + j], parity);
                tc_fence_after();
                tmem_ld_32x32(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + accp * kAccCols + kFinCol + 64 * j + 32 * hsel, r[j]);
            }
            if (lane == 0) tma_store_wait_read<0>();           // this warp's previous boxes have left the staging buffers
            tmem_ld_wait();
            __syncwarp();
            const uint32_t bias_c = bias_u32 + 4u * (64 + 32 * hsel);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {                   // one bias fetch serves both super-tiles (the kernel is bound by
                const float4 b0 = lds_f4(bias_c + 32u * jj), b1 = lds_f4(bias_c + 32u * jj + 16u);   // shared-memory wavefronts)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    uint32_t o[4];
                    o[0] = act_pack_t<ACT, FMT>(__uint_as_float(r[j][8 * jj]) + b0.x, __uint_as_float(r[j][8 * jj + 1]) + b0.y);
                    o[1] = act_pack_t<ACT, FMT>(__uint_as_float(r[j][8 * jj + 2]) + b0.z, __uint_as_float(r[j][8 * jj + 3]) + b0.w);
                    o[2] = act_pack_t<ACT, FMT>(__uint_as_float(r[j][8 * jj + 4]) + b1.x, __uint_as_float(r[j][8 * jj + 5]) + b1.y);
                    o[3] = act_pack_t<ACT, FMT>(__uint_as_float(r[j][8 * jj + 6]) + b1.z, __uint_as_float(r[j][8 * jj + 7]) + b1.w);
                    sts_u4(chain_stg + j * 2048 + lane * 64 + ((jj ^ ((lane >> 1) & 3)) << 4), o[0], o[1], o[2], o[3]);
                }
            }
            if (quad < 3) {
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) {
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                        if ((s_prev + j) * kChainRows < p.M2)
                            tma_store_3d(&p.tmOut, chain_stg + j * 2048, 32 * hsel, (s_prev + j) * kChainRows + quad * 32, b_prev);
                    tma_store_commit();
                }
            } else {
                __syncwarp();
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int l = (s_prev + j) * kChainRows + row_in_tile;
                    if (row_in_tile < kChainRows && l < p.M2) {
                        uint8_t* dst = reinterpret_cast<uint8_t*>(p.out2) + ((static_cast<size_t>(b_prev) * p.M2 + l) * 64 + 32 * hsel) * 2;
#pragma unroll
                        for (int uq = 0; uq < 4; ++uq)
                            *reinterpret_cast<float4*>(dst + 16 * uq) = lds_f4(chain_stg + j * 2048 + lane * 64 + ((uq ^ ((lane >> 1) & 3)) << 4));
                    }
                }
                __syncwarp();                                  // the buffers are rewritten in the next call
            }
        };
        int prev_batch = 0, prev_mt = 0;                       // EPI_FINAL / EPI_CHAIN: the tile whose second chain is in flight
        // EPI_CHAIN: this layer's 32 biases stay in registers (every lane needs all of them for every tile; read from shared
        // memory they were 128 of the ~2600 shared-memory wavefronts per super-tile that bound the kernel)
        float chain_bias[EPI == EPI_CHAIN ? 32 : 1];
        // EPI_STORE with N a constant (32, 64, 128: whole-window DeepClean layers): a warp's chunk pair covers the same 64 (32)
        // columns in every stage -- 32 (4 cp + 2 hsel + which) mod N does not depend on cp -- so their biases are read once.  A
        // broadcast ld.shared.v4 costs four wavefronts of the shared-memory data stage (its 512 bytes of return traffic), and
        // per stage they were two thirds of the epilogue's wavefronts on the stage that bounds these layers.  Same for the 64
        // columns of EPI_FINAL.
        constexpr bool kStoreBiasRegs = EPI == EPI_STORE && NT != 0;
        float4 store_bias[kStoreBiasRegs ? 2 : 1][kStoreBiasRegs ? 8 : 1];
        if (kStoreBiasRegs) {
#pragma unroll
            for (int which = 0; which < 2; ++which)
#pragma unroll
                for (int j = 0; j < 8; ++j) store_bias[which][j] = lds_f4(bias_u32 + 4u * (ch_col[which] + 4 * j));
        }
        float4 final_bias[EPI == EPI_FINAL ? 16 : 1];
        if (EPI == EPI_FINAL) {
#pragma unroll
            for (int j = 0; j < 16; ++j) final_bias[j] = lds_f4(bias_u32 + 16u * j);
        }
        if (EPI == EPI_CHAIN) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float4 b4 = lds_f4(bias_u32 + 16u * i);
                chain_bias[4 * i] = b4.x; chain_bias[4 * i + 1] = b4.y; chain_bias[4 * i + 2] = b4.z; chain_bias[4 * i + 3] = b4.w;
            }
        }
        const uint32_t stage_u32 = smem_u32(smem_out) + (warp - 2) * 4096;   // + 32 KiB for the second buffer
        int ostep = 0;
        int it = 0;
        TR_DECL
        for (int w = worker; w < total; w += n_workers, ++it) {
            const int u = p.reverse ? total - 1 - w : w;
            const int acc = it & 1;
            const int batch = (u / spi) * p.n_det + det;
            TR_WAIT(0, mbar_wait(&tmem_full[acc], (it >> 1) & 1))
            tc_fence_after();
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * kAccCols;
            if (EPI == EPI_STORE) {
                // 8 chunks of 32 columns per stage; this warp takes the adjacent chunk pairs (4 cp + 2 hsel, +1).
                // The activated 16-bit values go to this warp's staging buffer in the swizzled layout the
                // output tensor map expects (conflict-free 16-byte stores) and leave with ONE TMA store per
                // 32-row x 128-byte box (per-lane row stores would touch 32 lines with 16 bytes each per
                // instruction: measured 65 % L1TEX utilisation and ~60 % of HBM rate on the thin layers).
                // Rows past M are clipped by the tensor map.
                const bool wide = pN >= 64;
                for (int cp = 0; cp < 2; ++cp) {
                    const int ca = 4 * cp + 2 * hsel, cbk = ca + 1;              // chunk indices
                    // zone launches: does this warp's quadrant of the chunk's tile hold a recomputed row at all?
                    const int vta = (u % spi) * G + ch_g[2 * cp], vtb = (u % spi) * G + ch_g[2 * cp + 1];
                    const bool la = ch_g[2 * cp] < G && vta < p.v_tiles && quad_live(vta);
                    const bool lb = wide ? la : (ch_g[2 * cp + 1] < G && vtb < p.v_tiles && quad_live(vtb));
                    if (!la && !lb) {
                        if (cp == 1) {                         // nothing read from this stage by this warp: hand it back
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(&tmem_empty[acc]);
                        }
                        continue;
                    }
                    uint32_t ra[32], rb[32];
                    tmem_ld_32x32(taddr + 32 * ca, ra);
                    tmem_ld_32x32(taddr + 32 * cbk, rb);
                    float4 bia[2][8];                          // bias of both chunks, fetched under the TMEM latency
                    if (NT == 0) {
#pragma unroll
                        for (int which = 0; which < 2; ++which)
#pragma unroll
                            for (int j = 0; j < 8; ++j) bia[which][j] = lds_f4(bias_u32 + 4u * (ch_col[2 * cp + which] + 4 * j));
                    }
                    const uint32_t stg = stage_u32 + ((ostep % p.out_bufs) << 15);
                    if (lane == 0) {                           // the store that last read this buffer has drained it
                        TR_WAIT(1, if (p.out_bufs == 2) tma_store_wait_read<1>(); else tma_store_wait_read<0>())
                    }
                    ++ostep;
                    tmem_ld_wait();
                    if (cp == 1) {                             // last reads of this stage: hand it back
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&tmem_empty[acc]);
                    }
                    __syncwarp();
#pragma unroll
                    for (int which = 0; which < 2; ++which) {
                        const uint32_t* r = which == 0 ? ra : rb;
#pragma unroll
                        for (int jj = 0; jj < 4; ++jj) {       // 16-byte units of this chunk's 64-byte row
                            uint32_t o[4];
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const float4 b4 = NT ? store_bias[which][2 * jj + h] : bia[which][2 * jj + h];
                                o[2 * h] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h]) + b4.x, __uint_as_float(r[8 * jj + 4 * h + 1]) + b4.y);
                                o[2 * h + 1] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h + 2]) + b4.z, __uint_as_float(r[8 * jj + 4 * h + 3]) + b4.w);
                            }
                            const uint32_t addr = wide ? stg + lane * 128 + (((4 * which + jj) ^ (lane & 7)) << 4)
                                                       : stg + which * 2048 + lane * 64 + ((jj ^ ((lane >> 1) & 3)) << 4);
                            sts_u4(addr, o[0], o[1], o[2], o[3]);
                        }
                    }
                    fence_proxy_async();
                    __syncwarp();
                    {
                        const int row0 = quad * 32;
                        if (wide) {                            // both chunks: one tile, 64 adjacent columns
                            if (la) store_box(stg, ch_col[2 * cp], map_tile(p, vta) * kTileM + row0, batch, 128);
                        } else {                               // N = 32: the chunks are two consecutive tiles
                            if (la) store_box(stg, 0, map_tile(p, vta) * kTileM + row0, batch, 64);
                            if (lb) store_box(stg + 2048, 0, map_tile(p, vtb) * kTileM + row0, batch, 64);
                        }
                        if (lane == 0) tma_store_commit();
                    }
                }
            } else if (EPI == EPI_CHAIN) {
                // N = 32, four tiles per stage = two super-tiles: tile g holds positions chain_m0(vt) + [0, 128) of this layer
                // x 32 channels; this warp drains tiles g = hsel and hsel + 2 (super-tile j = 0, 1 of the stage).  Position
                // pair r of a super-tile (the next layer's A row r = 64 (g & 1) + position / 2) takes the position's 64 bytes
                // in its even or odd half.  Zero outside this layer's rows (the next layer's padding).
                const int s_cur = (u % spi) * 2;               // first super-tile of the stage
                uint32_t ra[2][32];
                tmem_ld_32x32(taddr + 32 * hsel, ra[0]);
                tmem_ld_32x32(taddr + 32 * (hsel + 2), ra[1]);
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tmem_empty[acc]);
                const int arow = 64 * hsel + (row_in_tile >> 1);
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const int vt = (u % spi) * G + hsel + 2 * j;
                    const int pos = chain_m0(vt) + row_in_tile;
                    const bool inside = vt < p.v_tiles && pos >= 0 && pos < p.M;
                    const uint32_t row_u32 = smem_u32(smem_out) + (acc * 2 + j) * kChainTile + arow * 128;
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        uint32_t o[4];
#pragma unroll
                        for (int h = 0; h < 2; ++h)
#pragma unroll
                            for (int q = 0; q < 2; ++q)
                                o[2 * h + q] = act_pack_t<ACT, FMT>(__uint_as_float(ra[j][8 * jj + 4 * h + 2 * q]) + chain_bias[8 * jj + 4 * h + 2 * q],
                                                                    __uint_as_float(ra[j][8 * jj + 4 * h + 2 * q + 1]) + chain_bias[8 * jj + 4 * h + 2 * q + 1]);
                        if (!inside) o[0] = o[1] = o[2] = o[3] = 0u;
                        sts_u4(row_u32 + ((((row_in_tile & 1) * 4 + jj) ^ (arow & 7)) << 4), o[0], o[1], o[2], o[3]);
                    }
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) { mbar_arrive(&stg_full[acc * 2]); mbar_arrive(&stg_full[acc * 2 + 1]); }
                if (it > 0) chain_emit(acc ^ 1, ((it - 1) >> 1) & 1, prev_batch, prev_mt);
                prev_batch = batch; prev_mt = s_cur;
            } else if (EPI == EPI_FINAL) {
                // N = 64, two tiles per stage: accumulator row i of tile g is input position m = mt * 126 - 1 + i of
                // this layer and holds its outputs x[2m][0..32) | x[2m+1][0..32) = one 128-byte row of the last
                // layer's A operand.  Warp (quad, hsel) activates rows [32 quad, +32) of tile g = hsel, writes them
                // (16-bit, zero outside the window = the last layer's padding) into the shared-memory tile
                // [acc][hsel] in the swizzled K-major layout and hands the tile to the MMA warp; the last layer
                //   y[4m + r] = b + sum_{a, par, ci} w[ci][r + 3 - 4a - 2 par] x[2(m + a) + par][ci],  a = -1, 0, 1,
                // is then three row-shifted K blocks on the tensor core (D3).  The 4 results of the
                // PREVIOUS tile are read back one iteration later, when its chain has long retired.
                const int vt = (u % spi) * G + hsel;
                const int mt = vt < p.v_tiles ? map_tile(p, vt) : p.tiles_m;   // tiles_m: no such tile
                // zone launches: this warp's 32 rows matter only if one of them, or a neighbour the second chain reads with
                // it, is a recomputed row (the first z_left / last z_right rows of the layer); else the stale shared-memory
                // rows stay and feed nothing but outputs that are not stored
                const int qr0 = mt * p.tile_stride + p.tile_row0 + quad * 32;
                const bool qlive = (z_left | z_right) == 0 || qr0 < z_left + 1 || qr0 + 32 > p.M - z_right - 1;
                uint32_t ra[32], rb[32];
                if (qlive) {
                    tmem_ld_32x32(taddr + 64 * hsel, ra);
                    tmem_ld_32x32(taddr + 64 * hsel + 32, rb);
                    tmem_ld_wait();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tmem_empty[acc]);
                const int row = mt * p.tile_stride + p.tile_row0 + row_in_tile;
                const bool inside = mt < p.tiles_m && row >= 0 && row < p.M;
                const uint32_t tile_u32 = smem_u32(smem_out) + (acc * 2 + hsel) * kFinTile + quad * 4096;
                if (qlive) {
#pragma unroll
                    for (int which = 0; which < 2; ++which) {
                        const uint32_t* r = which == 0 ? ra : rb;
#pragma unroll
                        for (int jj = 0; jj < 4; ++jj) {
                            uint32_t o[4];
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const float4 b4 = final_bias[8 * which + 2 * jj + h];
                                o[2 * h] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h]) + b4.x, __uint_as_float(r[8 * jj + 4 * h + 1]) + b4.y);
                                o[2 * h + 1] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h + 2]) + b4.z, __uint_as_float(r[8 * jj + 4 * h + 3]) + b4.w);
                            }
                            if (!inside) o[0] = o[1] = o[2] = o[3] = 0u;
                            sts_u4(tile_u32 + lane * 128 + (((4 * which + jj) ^ (lane & 7)) << 4), o[0], o[1], o[2], o[3]);
                        }
                    }
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&stg_full[acc * 2 + hsel]);
                if (it > 0) {
                    const int accp = acc ^ 1;
                    TR_WAIT(2, mbar_wait(&fin_full[accp * 2 + hsel], ((it - 1) >> 1) & 1))
                    tc_fence_after();
                    uint32_t y[4];
                    tmem_ld_32x4(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + accp * kAccCols + kFinCol + hsel * kFinN, y);
                    tmem_ld_wait();
                    const int orow = prev_mt * p.tile_stride + row_in_tile;     // D row i = tile row i + 1
                    if (row_in_tile < p.tile_stride && prev_mt < p.tiles_m && orow < p.M && fin_row_live(orow)) {
                        int o4 = 4 * orow;                                      // window position of y[4 orow]
                        if (pred_ring) { o4 += ring_h; if (o4 >= 4 * p.M) o4 -= 4 * p.M; }   // ring slot (absolute index mod W)
                        *reinterpret_cast<float4*>(p.pred + static_cast<size_t>(prev_batch) * p.M * 4 + o4) =
                            make_float4(__uint_as_float(y[0]) + fin_bias, __uint_as_float(y[1]) + fin_bias,
                                        __uint_as_float(y[2]) + fin_bias, __uint_as_float(y[3]) + fin_bias);
                    }
                }
                prev_batch = batch; prev_mt = mt;
            } else {
                // conv (stride 1) + bias + ReLU + MaxPool(4): row m holds outputs 2m (cols [0,N/2)) and 2m+1
                // (cols [N/2,N)); pooled row q = m/2 is the max over both halves of rows 2q and 2q+1.
                const int m0 = (u % spi) * kTileM;
                const int row = m0 + row_in_tile;
                const int half = pN / 2;
                const int Mq = p.M / 2;
                const int pstride = half + 1;
                float* pool_s = head_s;                        // [64][half+1] fp32 (EPI_POOL_HEAD only)
                const int n_chunks = half / 32;
                for (int ci = hsel; ci < n_chunks; ci += 2) {
                    const int c0 = ci * 32;
                    uint32_t re[32], ro[32];
                    tmem_ld_32x32(taddr + c0, re);
                    tmem_ld_32x32(taddr + half + c0, ro);
                    tmem_ld_wait();
                    float v[32];
#pragma unroll
                    for (int j = 0; j < 32; ++j) {
                        const float bj = bias_s[c0 + j];
                        float m = fmaxf(__uint_as_float(re[j]) + bj, __uint_as_float(ro[j]) + bj);
                        m = (row < p.M) ? fmaxf(m, 0.f) : 0.f;               // ReLU; rows past the end contribute 0
                        const float other = __shfl_xor_sync(0xffffffffu, m, 1);
                        v[j] = fmaxf(m, other);
                    }
                    if ((lane & 1) == 0 && row < p.M) {
                        const int q = row / 2;
                        if (EPI == EPI_POOL) {
                            uint16_t* orow = reinterpret_cast<uint16_t*>(p.out) + (static_cast<size_t>(batch) * Mq + q) * half + c0;
                            uint4* dst = reinterpret_cast<uint4*>(orow);
#pragma unroll
                            for (int j = 0; j < 4; ++j)
                                dst[j] = make_uint4(pack_pair_t<FMT>(v[8 * j], v[8 * j + 1]), pack_pair_t<FMT>(v[8 * j + 2], v[8 * j + 3]),
                                                    pack_pair_t<FMT>(v[8 * j + 4], v[8 * j + 5]), pack_pair_t<FMT>(v[8 * j + 6], v[8 * j + 7]));
                        } else {
                            float* prow = pool_s + (row_in_tile / 2) * pstride + c0;
#pragma unroll
                            for (int j = 0; j < 32; ++j) prow[j] = v[j];
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tmem_empty[acc]);
                if (EPI == EPI_POOL_HEAD) {
                    // global average pool over the Mq pooled rows, dense(half -> hidden) + ReLU,
                    // dense(hidden -> 1), sigmoid: fused into this (last) conv block's epilogue.
                    float* gap_s = pool_s + 64 * pstride;                    // [half]
                    float* hid_s = gap_s + half;                             // [hidden]
                    // this warp's rows of the first dense layer (hidden <= 64, half <= 128: 8 rows x 4 values per lane),
                    // requested NOW so that their L2 latency runs under the pooling barriers instead of once per row
                    const bool pre_w = p.head_hidden <= 8 * kEpiWarps && half <= 128;
                    float wreg[8][4];
                    if (pre_w) {
#pragma unroll
                        for (int rr = 0; rr < 8; ++rr) {
                            const int hrow = warp - 2 + rr * kEpiWarps;
#pragma unroll
                            for (int k = 0; k < 4; ++k) {
                                const int c = lane + 32 * k;
                                wreg[rr][k] = (hrow < p.head_hidden && c < half) ? __ldg(p.hw1 + static_cast<size_t>(hrow) * half + c) : 0.f;
                            }
                        }
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");
                    for (int c = et; c < half; c += kEpiWarps * 32) {
                        float s = 0.f;
                        for (int q = 0; q < Mq; ++q) s += pool_s[q * pstride + c];
                        gap_s[c] = s / static_cast<float>(Mq);
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");
                    // one warp per hidden unit, lanes stride over the inputs: the weight row is read with coalesced
                    // 128-byte requests (one thread per row walked 128 dependent, uncoalesced loads: ~15 us per launch)
                    if (pre_w) {
                        float gv[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) gv[k] = lane + 32 * k < half ? gap_s[lane + 32 * k] : 0.f;
#pragma unroll
                        for (int rr = 0; rr < 8; ++rr) {
                            const int hrow = warp - 2 + rr * kEpiWarps;
                            float s = 0.f;
#pragma unroll
                            for (int k = 0; k < 4; ++k) s = fmaf(wreg[rr][k], gv[k], s);      // same order as the loop below
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                            if (lane == 0 && hrow < p.head_hidden) hid_s[hrow] = fmaxf(s + __ldg(p.hb1 + hrow), 0.f);
                        }
                    } else {
                        for (int hrow = warp - 2; hrow < p.head_hidden; hrow += kEpiWarps) {
                            const float* wr = p.hw1 + static_cast<size_t>(hrow) * half;
                            float s = 0.f;
                            for (int c = lane; c < half; c += 32) s = fmaf(__ldg(wr + c), gap_s[c], s);
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                            if (lane == 0) hid_s[hrow] = fmaxf(s + __ldg(p.hb1 + hrow), 0.f);
                        }
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");
                    if (et < 32) {
                        float s = 0.f;
                        for (int i = et; i < p.head_hidden; i += 32) s = fmaf(__ldg(p.hw2 + i), hid_s[i], s);
#pragma unroll
                        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
                        if (et == 0) {
                            const float z = s + __ldg(p.hb2);
                            p.scores[batch] = 1.f / (1.f + __expf(-z));
                        }
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");           // scratch is reused by the next tile
                }
            }
        }
        if (EPI == EPI_CHAIN && it > 0) chain_emit((it - 1) & 1, ((it - 1) >> 1) & 1, prev_batch, prev_mt);
        if (EPI == EPI_FINAL && it > 0) {                      // the last tile's second chain
            const int accp = (it - 1) & 1;
            mbar_wait(&fin_full[accp * 2 + hsel], ((it - 1) >> 1) & 1);
            tc_fence_after();
            uint32_t y[4];
            tmem_ld_32x4(tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + accp * kAccCols + kFinCol + hsel * kFinN, y);
            tmem_ld_wait();
            const int orow = prev_mt * p.tile_stride + row_in_tile;
            if (row_in_tile < p.tile_stride && prev_mt < p.tiles_m && orow < p.M && fin_row_live(orow)) {
                int o4 = 4 * orow;
                if (pred_ring) { o4 += ring_h; if (o4 >= 4 * p.M) o4 -= 4 * p.M; }
                *reinterpret_cast<float4*>(p.pred + static_cast<size_t>(prev_batch) * p.M * 4 + o4) =
                    make_float4(__uint_as_float(y[0]) + fin_bias, __uint_as_float(y[1]) + fin_bias,
                                __uint_as_float(y[2]) + fin_bias, __uint_as_float(y[3]) + fin_bias);
            }
        }
        if (warp == 2) { TR_FLUSH(8, 3) }
    }
    if ((EPI == EPI_STORE || EPI == EPI_CHAIN) && warp >= 2 && warp < kMmaWarp2 && lane == 0) tma_store_wait_all<0>();   // staging buffers are still being read
    tc_fence_before();
    __syncthreads();
    stamp_end(p.stamp);
    if (warp == 0) tmem_dealloc(tmem_base, 2 * kAccCols);
}

// ---------------------------------------------------------------------------------------------
// CTA-pair variant for the layers whose weights do not fit in shared memory (GEMM N = 256, EPI_STORE).
//
// With one CTA per tile such a layer is bound by SHARED-MEMORY bandwidth, not by the tensor pipe: per
// 128 x 256 x 896 tile the tensor core reads 56 x (4 KiB A + 8 KiB B), TMA writes 448 KiB of weights and 67 KiB
// of slabs, the epilogue moves 128 KiB -- 1.3 MiB at 128 B/clk = 10.3 k cycles against 7.2 k cycles of math
// (measured 13.5 k; profiles/r01_mma_rate_microbench.txt).  Here two CTAs of a cluster (one TPC) work on two
// consecutive tiles as ONE tcgen05.mma.cta_group::2 of M = 256: each CTA loads its own A slab but only HALF of
// every weight block (128 of the 256 rows of B), and the tensor cores of both SMs read both halves.  Weight
// fills and weight reads per SM halve (1.3 MiB -> 0.85 MiB per tile).
//
// Roles per CTA (320 threads): warp 0 TMA producer (both CTAs; completion bytes are counted on the LEADER's
// barriers), warp 1 MMA issuer (leader only; commits multicast to both CTAs), warps 2-9 epilogue (each CTA
// drains its own 128 TMEM lanes; the peer's warps release the accumulator stage on the leader's barrier).
// ---------------------------------------------------------------------------------------------
constexpr int kGemm2Threads = 64 + kEpiWarps * 32;
constexpr int kHalfB = 128 * 128;                    // half of one weight K block: 128 rows x 128 bytes

// PACKED is a template parameter so that the whole-window instantiation (the two heaviest launches of the full step)
// compiles without a trace of the zone packing: with the packing as a run-time branch it took 164 registers instead of 151
// and ran 15 % slower per cycle.
template <int ACT, int FMT, bool PACKED>
__global__ void __launch_bounds__(kGemm2Threads, 1) k_conv_gemm_2sm(const __grid_constant__ ConvGemmParams p, int n_items) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    // Packed zones (incremental path, p.pk_nl > 0): a tile holds both recomputed zones of pk_k consecutive batch items, one
    // segment of pk_seg = pk_nl + pk_nr rows each -- slab rows [0, pk_nl) of a segment are the input rows of the left zone
    // (outputs 0 .. pk_left-1), the next pk_nr rows those of the right zone (tile rows pk_nl .. pk_nl + pk_right - 1 of the
    // segment = the layer's LAST pk_right rows); the tile rows in between mix neighbours and are dropped.  The two CTAs
    // of a pair then work on 2 pk_k consecutive batch items.
    constexpr bool packed = PACKED;
    const int sl = slab_bytes_of(p.slab_rows + (PACKED ? p.pk_nl : 0));
    const int sa = p.sa_stages, sb = p.sb_stages;
    uint8_t* smem_out = smem;                                                // [out_bufs][8 warps][4 KiB]
    uint8_t* smem_b = smem + p.out_bufs * kOutStage;                         // [sb][16 KiB]
    uint8_t* smem_a = smem_b + sb * kHalfB;                                  // [sa][slab]
    uint8_t* after_a = smem_a + sa * sl;
    float* bias_s = reinterpret_cast<float*>(after_a);                       // [256]
    uint64_t* bars = reinterpret_cast<uint64_t*>(after_a + 1024);
    uint64_t* a_full = bars;                 // [8]  leader's are used
    uint64_t* a_empty = a_full + 8;          // [8]
    uint64_t* b_full = a_empty + 8;          // [8]  leader's are used
    uint64_t* b_empty = b_full + 8;          // [8]
    uint64_t* tmem_full = b_empty + 8;       // [2]
    uint64_t* tmem_empty = tmem_full + 2;    // [2]  leader's are used: 2 x 8 epilogue warps arrive
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    stamp_begin(p.stamp);
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x / 32, 0);
    const int lane = threadIdx.x % 32;
    const uint32_t rank = cluster_ctarank();                                 // 0 = leader
    const int cid = blockIdx.x / 2;
    const int det = cid % p.n_det;
    const int cworker = cid / p.n_det;
    const int n_cw = (gridDim.x / 2) / p.n_det;
    const int half_tiles = packed ? 1 : p.v_tiles / 2;                       // (virtual) tile pairs per batch item
    const int pk_seg = PACKED ? p.pk_nl + p.pk_nr : 1;
    const int total = packed ? n_items / (2 * p.pk_k) : n_items * half_tiles; // packed: one pair = 2 pk_k batch items

    if (warp == 0) {
        if (lane == 0) {
            tma_prefetch_desc(&p.tmA);
            tma_prefetch_desc(&p.tmB);
            for (int i = 0; i < 8; ++i) {
                mbar_init(&a_full[i], 1); mbar_init(&a_empty[i], 1);
                mbar_init(&b_full[i], 1); mbar_init(&b_empty[i], 1);
            }
            for (int i = 0; i < 2; ++i) { mbar_init(&tmem_full[i], 1); mbar_init(&tmem_empty[i], 2 * kEpiWarps); }
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc_2sm(tmem_slot, 2 * kAccCols);
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                          // both CTAs' barriers exist before anything arrives on them
    tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);
    griddep_launch_dependents();

    if (warp == 0) {
        // --------------------------------------------------------------- TMA producer (both CTAs)
        // Two cursors.  The WEIGHT cursor walks the flat schedule (work item, segment 0 .. n_seg-1; segment order
        // is issue order, `cbstart` marks the first segment of a column block) and blocks on b_empty.  The SLAB
        // cursor runs ahead of it without blocking (a stage frees up a whole tile before its next use), and is
        // only forced -- blocking -- to have issued slab (item, cb) before the first weight block of that column
        // block (otherwise the weight ring could fill while the MMA warp waits for the slab).
        griddep_wait();
        // ring input: this update's window has its own tensor map (rows outside the window are zero fill)
        const int head = p.tmA_heads ? static_cast<int>(*p.a_count % p.a_ring_W) / p.head_div : 0;
        const CUtensorMap* tmA = p.tmA_heads ? p.tmA_heads + head : &p.tmA;
        const CUtensorMap* tmA_left = packed ? p.tmA_heads_left + head : nullptr;   // box of pk_nl rows
        const CUtensorMap* tmA_right = packed ? p.tmA_heads_right + head : nullptr; // box of pk_nr rows
        const uint32_t lead_a_full = mapa_u32(smem_u32(a_full), 0), lead_b_full = mapa_u32(smem_u32(b_full), 0);
        unsigned long long cbstart = 0;
        {
            int sidx = 0;
            for (int cb = 0; cb < p.n_cb; ++cb) {
                bool first = true;
                for (int sh = 0; sh < p.n_shift; ++sh)
                    if (p.seg_of[cb][sh] >= 0) { if (first) cbstart |= 1ull << sidx; first = false; ++sidx; }
            }
        }
        const int n_cb = p.n_cb, n_seg = p.n_seg;
        int stage = 0; uint32_t aph = 0;
        int bs = 0; uint32_t bph = 0;
        int aw = cworker, acb = 0;                                           // slab cursor: work item, column block
        int a_issued = 0, a_needed = 0;                                      // slabs issued / slabs the weight cursor requires
        TR_DECL
        auto slab_step = [&](bool block) -> bool {                           // issue the slab under the cursor, if it can be
            if (aw >= total) return false;
            if (block) { TR_WAIT(0, mbar_wait(&a_empty[stage], aph ^ 1)) }
            else if (!__shfl_sync(0xffffffffu, mbar_test_wait(&a_empty[stage], aph ^ 1) ? 1 : 0, 0)) return false;
            if (lane == 0) {
                const int u = p.reverse ? total - 1 - aw : aw;
                if (packed) {
                    if (rank == 0) mbar_arrive_expect_tx(&a_full[stage], 2 * p.pk_k * pk_seg * 128);
                    for (int w = 0; w < p.pk_k; ++w) {
                        const int batch = ((2 * u + static_cast<int>(rank)) * p.pk_k + w) * p.n_det + det;
                        uint8_t* seg = smem_a + stage * sl + w * pk_seg * 128;
                        tma_load_3d_2sm(seg, tmA_left, lead_a_full + 8u * stage, acb * kSegK, p.a_min, batch);
                        tma_load_3d_2sm(seg + p.pk_nl * 128, tmA_right, lead_a_full + 8u * stage, acb * kSegK,
                                        p.M - p.pk_right + p.a_min, batch);
                    }
                } else {
                    const int m0 = map_tile(p, (u % half_tiles) * 2 + static_cast<int>(rank)) * kTileM;
                    if (rank == 0) mbar_arrive_expect_tx(&a_full[stage], 2 * p.slab_rows * 128);
                    tma_load_3d_2sm(smem_a + stage * sl, tmA, lead_a_full + 8u * stage, acb * kSegK, m0 + p.a_min,
                                    (u / half_tiles) * p.n_det + det);
                }
            }
            if (++stage == sa) { stage = 0; aph ^= 1; }
            if (++acb == n_cb) { acb = 0; aw += n_cw; }
            ++a_issued;
            return true;
        };
        for (int w = cworker; w < total; w += n_cw) {
            for (int sg = 0; sg < n_seg; ++sg) {
                if ((cbstart >> sg) & 1ull) {
                    ++a_needed;
                    while (a_issued < a_needed) slab_step(true);
                }
                while (slab_step(false)) {}
                TR_WAIT(1, mbar_wait(&b_empty[bs], bph ^ 1))
                if (lane == 0) {
                    if (rank == 0) mbar_arrive_expect_tx(&b_full[bs], 2 * kHalfB);
                    tma_load_3d_2sm(smem_b + bs * kHalfB, &p.tmB, lead_b_full + 8u * bs, sg * kSegK, static_cast<int>(rank) * 128, det);
                }
                if (++bs == sb) { bs = 0; bph ^= 1; }
            }
        }
        TR_FLUSH(0, 2)
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer (leader CTA)
        if (rank == 0) {
            const uint32_t idesc = umma_idesc_f16(FMT, 2 * kTileM, 256);
            const uint32_t smem_a_u32 = smem_u32(smem_a), smem_b_u32 = smem_u32(smem_b);
            const int n_cb = p.n_cb, n_shift = p.n_shift;
            unsigned long long shmask = 0;
            for (int cb = 0; cb < n_cb; ++cb)
                for (int sh = 0; sh < n_shift; ++sh)
                    if (p.seg_of[cb][sh] >= 0) shmask |= 1ull << (cb * kMaxShift + sh);
            const uint32_t leader = elect_one() ? 1u : 0u;
            int it = 0;
            TR_DECL
            int stage = 0; uint32_t aph = 0;
            int bs = 0; uint32_t bph = 0;
            for (int w = cworker; w < total; w += n_cw, ++it) {
                const int acc = it & 1;
                TR_WAIT(0, mbar_wait(&tmem_empty[acc], ((it >> 1) & 1) ^ 1))
                tc_fence_after();
                const uint32_t d_tmem = tmem_base + acc * kAccCols;
                uint32_t accumulate = 0;
                for (int cb = 0; cb < n_cb; ++cb) {
                    const uint32_t m = static_cast<uint32_t>(shmask >> (cb * kMaxShift)) & ((1u << kMaxShift) - 1);
                    TR_WAIT(1, mbar_wait(&a_full[stage], aph))
                    tc_fence_after();
                    const uint32_t a_lo = umma_desc_lo(smem_a_u32 + stage * sl);
                    for (int sh = 0; sh < n_shift; ++sh) {
                        if (!((m >> sh) & 1u)) continue;
                        TR_WAIT(2, mbar_wait(&b_full[bs], bph))
                        tc_fence_after();
                        const uint32_t bl = umma_desc_lo(smem_b_u32 + bs * kHalfB);
                        const uint32_t a_lo_s = a_lo + 8u * sh;
#pragma unroll
                        for (int k = 0; k < kSegK / 16; ++k)
                            umma_f16_2sm_if(leader, d_tmem, umma_desc_make(a_lo_s + 2 * k), umma_desc_make(bl + 2 * k), idesc, accumulate | k);
                        umma_commit_2sm_if(leader, &b_empty[bs]);
                        if ((m >> (sh + 1)) == 0) umma_commit_2sm_if(leader, &a_empty[stage]);
                        accumulate = 1;
                        if (++bs == sb) { bs = 0; bph ^= 1; }
                    }
                    if (++stage == sa) { stage = 0; aph ^= 1; }
                }
                umma_commit_2sm_if(leader, &tmem_full[acc]);
            }
            TR_FLUSH(3, 4)
        }
    } else {
        // ----------------------------------------------- epilogue warps 2..9 (both CTAs, own 128 TMEM lanes)
        const int quad = warp % 4;
        const int hsel = (warp - 2) / 4;
        const int et = threadIdx.x - 64;
        for (int i = et; i < 256; i += kEpiWarps * 32) bias_s[i] = __ldg(p.bias + static_cast<size_t>(det) * 256 + i);
        asm volatile("bar.sync 1, 256;" ::: "memory");
        const uint32_t bias_u32 = smem_u32(bias_s);
        griddep_wait();
        const int out_off = p.out_ring_div ? static_cast<int>(*p.a_count % p.a_ring_W) / p.out_ring_div : 0;
        const uint32_t stage_u32 = smem_u32(smem_out) + (warp - 2) * 4096;
        const uint32_t empty_addr[2] = {mapa_u32(smem_u32(&tmem_empty[0]), 0), mapa_u32(smem_u32(&tmem_empty[1]), 0)};
        int ostep = 0;
        int it = 0;
        TR_DECL
        for (int w = cworker; w < total; w += n_cw, ++it) {
            const int u = p.reverse ? total - 1 - w : w;
            const int acc = it & 1;
            const int batch = packed ? 0 : (u / half_tiles) * p.n_det + det;      // packed: per segment, below
            const int mt = packed ? 0 : map_tile(p, (u % half_tiles) * 2 + static_cast<int>(rank));
            TR_WAIT(0, mbar_wait(&tmem_full[acc], (it >> 1) & 1))
            tc_fence_after();
            const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16) + acc * kAccCols;
            if (packed) {
                // this lane's tile row: a row of the left zone, of the right zone, or one of the mixed rows in between;
                // the few live rows go straight from registers to their ring row and its twin (r +- M)
                const int i = quad * 32 + lane;
                const int w = i / pk_seg, j = i - w * pk_seg;       // segment (batch item of this CTA) and row inside it
                const int lrow = w >= p.pk_k ? -1 : j < p.pk_left ? j
                               : (j >= p.pk_nl && j < p.pk_nl + p.pk_right) ? p.M - p.pk_right + j - p.pk_nl : -1;
                const int pbatch = ((2 * u + static_cast<int>(rank)) * p.pk_k + w) * p.n_det + det;
                const int r = out_off + lrow, r2 = r >= p.M ? r - p.M : r + p.M;
                uint8_t* row1 = reinterpret_cast<uint8_t*>(p.out) + (static_cast<size_t>(pbatch) * 2 * p.M + r) * 512;
                uint8_t* row2 = reinterpret_cast<uint8_t*>(p.out) + (static_cast<size_t>(pbatch) * 2 * p.M + r2) * 512;
                for (int cp = 0; cp < 2; ++cp) {
                    const int col = 32 * (4 * cp + 2 * hsel);
                    uint32_t ra[32], rb[32];
                    tmem_ld_32x32(taddr + col, ra);
                    tmem_ld_32x32(taddr + col + 32, rb);
                    tmem_ld_wait();
                    if (cp == 1) {
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive_cluster(empty_addr[acc]);
                    }
                    if (lrow >= 0) {
#pragma unroll
                        for (int which = 0; which < 2; ++which) {
                            const uint32_t* rr = which == 0 ? ra : rb;
#pragma unroll
                            for (int jj = 0; jj < 4; ++jj) {
                                uint32_t o[4];
#pragma unroll
                                for (int h = 0; h < 2; ++h) {
                                    const float4 b4 = lds_f4(bias_u32 + 4u * (col + 32 * which + 8 * jj + 4 * h));
                                    o[2 * h] = act_pack_t<ACT, FMT>(__uint_as_float(rr[8 * jj + 4 * h]) + b4.x, __uint_as_float(rr[8 * jj + 4 * h + 1]) + b4.y);
                                    o[2 * h + 1] = act_pack_t<ACT, FMT>(__uint_as_float(rr[8 * jj + 4 * h + 2]) + b4.z, __uint_as_float(rr[8 * jj + 4 * h + 3]) + b4.w);
                                }
                                const int off = (col + 32 * which + 8 * jj) * 2;
                                *reinterpret_cast<uint4*>(row1 + off) = make_uint4(o[0], o[1], o[2], o[3]);
                                *reinterpret_cast<uint4*>(row2 + off) = make_uint4(o[0], o[1], o[2], o[3]);
                            }
                        }
                    }
                }
                continue;
            }
            for (int cp = 0; cp < 2; ++cp) {
                const int col = 32 * (4 * cp + 2 * hsel);                    // 64 adjacent columns: two 32-column chunks
                uint32_t ra[32], rb[32];
                tmem_ld_32x32(taddr + col, ra);
                tmem_ld_32x32(taddr + col + 32, rb);
                float4 bia[2][8];
#pragma unroll
                for (int which = 0; which < 2; ++which)
#pragma unroll
                    for (int j = 0; j < 8; ++j) bia[which][j] = lds_f4(bias_u32 + 4u * (col + 32 * which + 4 * j));
                const uint32_t stg = stage_u32 + ((ostep % p.out_bufs) << 15);
                if (lane == 0) {
                    TR_WAIT(1, if (p.out_bufs == 2) tma_store_wait_read<1>(); else tma_store_wait_read<0>())
                }
                ++ostep;
                tmem_ld_wait();
                if (cp == 1) {                                               // stage drained: tell the leader's MMA warp
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(empty_addr[acc]);
                }
                __syncwarp();
#pragma unroll
                for (int which = 0; which < 2; ++which) {
                    const uint32_t* r = which == 0 ? ra : rb;
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        uint32_t o[4];
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const float4 b4 = bia[which][2 * jj + h];
                            o[2 * h] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h]) + b4.x, __uint_as_float(r[8 * jj + 4 * h + 1]) + b4.y);
                            o[2 * h + 1] = act_pack_t<ACT, FMT>(__uint_as_float(r[8 * jj + 4 * h + 2]) + b4.z, __uint_as_float(r[8 * jj + 4 * h + 3]) + b4.w);
                        }
                        sts_u4(stg + lane * 128 + (((4 * which + jj) ^ (lane & 7)) << 4), o[0], o[1], o[2], o[3]);
                    }
                }
                fence_proxy_async();
                __syncwarp();
                {
                    // mirror ring (incremental path): ring row r and its twin r +- M; see store_box in k_conv_gemm_umma
                    const int r = out_off + mt * kTileM + quad * 32;
                    if (lane == 0) {
                        tma_store_3d(&p.tmOut, stg, col, r, batch);
                        if (p.out_ring_div) {
                            if (r >= p.M) tma_store_3d(&p.tmOut, stg, col, r - p.M, batch);
                            else tma_store_3d(&p.tmOut, stg, col, r + p.M, batch);
                        }
                        tma_store_commit();
                    }
                    if (p.out_ring_div && r < p.M && r + 31 >= p.M && r + lane >= p.M) {
                        uint8_t* dst = reinterpret_cast<uint8_t*>(p.out) +
                                       ((static_cast<size_t>(batch) * 2 * p.M + (r + lane - p.M)) * p.N + col) * 2;
#pragma unroll
                        for (int uu = 0; uu < 8; ++uu)
                            *reinterpret_cast<float4*>(dst + 16 * uu) = lds_f4(stg + lane * 128 + ((uu ^ (lane & 7)) << 4));
                    }
                }
            }
        }
        if (lane == 0) tma_store_wait_all<0>();
        if (warp == 2) { TR_FLUSH(8, 3) }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                          // the peer may still be reading this CTA's shared memory / TMEM
    stamp_end(p.stamp);
    if (warp == 0) tmem_dealloc_2sm(tmem_base, 2 * kAccCols);
}

typedef void (*Gemm2Kernel)(const ConvGemmParams, int);
template <bool PACKED>
static Gemm2Kernel pick_kernel_2sm_t(int act, int fmt) {
    if (act == ACT_TANH) return fmt == FMT_BF16 ? k_conv_gemm_2sm<ACT_TANH, FMT_BF16, PACKED> : k_conv_gemm_2sm<ACT_TANH, FMT_FP16, PACKED>;
    if (act == ACT_RELU) return fmt == FMT_BF16 ? k_conv_gemm_2sm<ACT_RELU, FMT_BF16, PACKED> : k_conv_gemm_2sm<ACT_RELU, FMT_FP16, PACKED>;
    return fmt == FMT_BF16 ? k_conv_gemm_2sm<ACT_NONE, FMT_BF16, PACKED> : k_conv_gemm_2sm<ACT_NONE, FMT_FP16, PACKED>;
}
static Gemm2Kernel pick_kernel_2sm(int act, int fmt, bool packed) {
    return packed ? pick_kernel_2sm_t<true>(act, fmt) : pick_kernel_2sm_t<false>(act, fmt);
}

// ---------------------------------------------------------------------------------------------
// Diagnostic (gw_probe_mma_cycles): cycles per tcgen05.mma.cta_group::1.kind::f16 (M = 128, K = 16, both operands in
// shared memory, SWIZZLE_128B K-major) as a function of N, issued back to back by one warp of one CTA with the
// descriptor pattern of a conv layer (four row shifts x four K steps).  This is the measurement behind the
// shared-memory-operand roofline of DESIGN.md section 7: cycles = max(N/2, 32 + N/4).
// ---------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(128, 1) k_probe_mma(long long* out, int reps) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    __shared__ uint64_t bar;
    __shared__ uint32_t slot;
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    for (int i = threadIdx.x; i < 176 * 1024 / 4; i += 128) reinterpret_cast<uint32_t*>(smem)[i] = 0;
    if (warp == 0) {
        if (lane == 0) { mbar_init(&bar, 1); fence_barrier_init(); }
        __syncwarp();
        tmem_alloc(&slot, 512);
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = slot;
    if (warp == 1) {
        const uint32_t idesc = umma_idesc_f16(FMT_FP16, kTileM, N);
        const uint32_t a_lo = umma_desc_lo(smem_u32(smem));             // a slab of 131 rows
        const uint32_t b_lo = umma_desc_lo(smem_u32(smem + 32768));     // four K blocks of N rows
        const uint32_t leader = elect_one() ? 1u : 0u;
        const long long t0 = clock64();
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int sh = 0; sh < 4; ++sh)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    umma_f16_if(leader, tmem + (r & 1) * 256, umma_desc_make(a_lo + 8u * sh + 2 * k),
                                umma_desc_make(b_lo + static_cast<uint32_t>(sh * N * 128 >> 4) + 2 * k), idesc, 1u);
        }
        const long long t1 = clock64();
        umma_commit_if(leader, &bar);
        mbar_wait(&bar, 0);
        const long long t2 = clock64();
        if (lane == 0) { out[0] = t1 - t0; out[1] = t2 - t0; }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 512);
}

template <int N>
static cudaError_t probe_one(long long* d_out, int reps, float* issue, float* complete) {
    cudaError_t e = cudaFuncSetAttribute(k_probe_mma<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, 180 * 1024);
    if (e != cudaSuccess) return e;
    long long h[2] = {0, 0};
    for (int it = 0; it < 2; ++it) {                       // second run: instruction cache and clocks warm
        k_probe_mma<N><<<1, 128, 180 * 1024>>>(d_out, reps);
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) return e;
    }
    e = cudaMemcpy(h, d_out, sizeof h, cudaMemcpyDeviceToHost);
    *issue = static_cast<float>(h[0]) / (reps * 16.0f);
    *complete = static_cast<float>(h[1]) / (reps * 16.0f);
    return e;
}

cudaError_t probe_mma_cycles(int N, float* issue, float* complete) {
    long long* d_out = nullptr;
    cudaError_t e = cudaMalloc(&d_out, 16);
    if (e != cudaSuccess) return e;
    const int reps = 64;
    switch (N) {
        case 16: e = probe_one<16>(d_out, reps, issue, complete); break;
        case 32: e = probe_one<32>(d_out, reps, issue, complete); break;
        case 64: e = probe_one<64>(d_out, reps, issue, complete); break;
        case 128: e = probe_one<128>(d_out, reps, issue, complete); break;
        case 256: e = probe_one<256>(d_out, reps, issue, complete); break;
        default: e = cudaErrorInvalidValue;
    }
    cudaFree(d_out);
    return e;
}

typedef void (*GemmKernel)(const ConvGemmParams, int);

static GemmKernel pick_kernel(int epi, int act, int fmt, bool zone, int N = 0) {
    if (epi == EPI_CHAIN && act == ACT_TANH)
        return fmt == FMT_BF16 ? k_conv_gemm_umma<EPI_CHAIN, ACT_TANH, FMT_BF16, false, 32> : k_conv_gemm_umma<EPI_CHAIN, ACT_TANH, FMT_FP16, false, 32>;
    // whole-window DeepClean layers (store epilogue, tanh): N is a template parameter
    if (epi == EPI_STORE && act == ACT_TANH && !zone) {
        if (N == 32) return fmt == FMT_BF16 ? k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_BF16, false, 32> : k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_FP16, false, 32>;
        if (N == 64) return fmt == FMT_BF16 ? k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_BF16, false, 64> : k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_FP16, false, 64>;
        if (N == 128) return fmt == FMT_BF16 ? k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_BF16, false, 128> : k_conv_gemm_umma<EPI_STORE, ACT_TANH, FMT_FP16, false, 128>;
    }
#define GW_PICK(E, A)                                                                                         \
    if (epi == E && act == A)                                                                                 \
        return zone ? (fmt == FMT_BF16 ? k_conv_gemm_umma<E, A, FMT_BF16, true, 0> : k_conv_gemm_umma<E, A, FMT_FP16, true, 0>)   \
                    : (fmt == FMT_BF16 ? k_conv_gemm_umma<E, A, FMT_BF16, false, 0> : k_conv_gemm_umma<E, A, FMT_FP16, false, 0>);
    GW_PICK(EPI_STORE, ACT_TANH)
    GW_PICK(EPI_STORE, ACT_NONE)
    GW_PICK(EPI_STORE, ACT_RELU)
    GW_PICK(EPI_FINAL, ACT_TANH)
    GW_PICK(EPI_POOL, ACT_RELU)
    GW_PICK(EPI_POOL_HEAD, ACT_RELU)
#undef GW_PICK
    return nullptr;
}

static bool g_prepared = false;
cudaError_t conv_gemm_prepare() {
    if (g_prepared) return cudaSuccess;
    const int epis[6] = {EPI_STORE, EPI_STORE, EPI_STORE, EPI_POOL, EPI_POOL_HEAD, EPI_FINAL};
    const int acts[6] = {ACT_TANH, ACT_NONE, ACT_RELU, ACT_RELU, ACT_RELU, ACT_TANH};
    for (int i = 0; i < 6; ++i)
        for (int fmt = 0; fmt < 2; ++fmt) {
            for (int zone = 0; zone < 2; ++zone)
                for (int N = 0; N <= 128; N = N ? 2 * N : 32) {
                    cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void*>(pick_kernel(epis[i], acts[i], fmt, zone != 0, N)),
                                                         cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
                    if (e != cudaSuccess) return e;
                }
        }
    for (int fmt = 0; fmt < 2; ++fmt) {
        cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void*>(pick_kernel(EPI_CHAIN, ACT_TANH, fmt, false, 32)),
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
    }
    for (int act = 0; act < 3; ++act)
        for (int fmt = 0; fmt < 2; ++fmt) {
            for (int pk = 0; pk < 2; ++pk) {
                cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void*>(pick_kernel_2sm(act, fmt, pk != 0)),
                                                     cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
                if (e != cudaSuccess) return e;
            }
        }
    g_prepared = true;
    return cudaSuccess;
}

cudaError_t launch_conv_gemm_umma(const GemmLaunch& g, cudaStream_t st) {
    const int n_items = g.batch / g.p.n_det;
    const int per_unit = g.p.epi == EPI_STORE ? (g.p.g_tiles ? g.p.g_tiles : kAccCols / g.p.N)
                                              : g.p.epi == EPI_CHAIN ? 4 : g.p.epi == EPI_FINAL ? 2 : 1;
    const int total = n_items * ((g.p.v_tiles + per_unit - 1) / per_unit);   // work units per detector
    int workers = g.grid / g.p.n_det;
    if (workers > total) workers = total;
    // the store epilogue without the zone forms is 9-11 % faster on e2 / e3 / d2 (measured, n = 128); the fused tail is
    // 5 % SLOWER without them (code placement), so it always runs the instantiation that has them (inert in whole windows)
    const bool zone = g.p.epi == EPI_FINAL || g.p.out_ring_div || g.p.pred_ring || g.p.z_left || g.p.z_right;
    GemmKernel k = pick_kernel(g.p.epi, g.p.act, g.p.fmt, zone, g.p.N);
    if (!k) return cudaErrorInvalidDeviceFunction;           // no kernel for this (epilogue, activation) pair
    cudaError_t e;
    if (g.p.two_sm) {
        int cw = g.grid / 2 / g.p.n_det;                         // clusters per detector
        const int units = g.p.pk_nl ? n_items / (2 * g.p.pk_k) : n_items * (g.p.v_tiles / 2);
        if (cw > units) cw = units;
        cudaLaunchConfig_t cfg2 = {};
        cfg2.gridDim = dim3(2 * cw * g.p.n_det);
        cfg2.blockDim = dim3(kGemm2Threads);
        cfg2.dynamicSmemBytes = g.smem_bytes;
        cfg2.stream = st;
        cudaLaunchAttribute at2[2];
        at2[0].id = cudaLaunchAttributeClusterDimension;
        at2[0].val.clusterDim.x = 2; at2[0].val.clusterDim.y = 1; at2[0].val.clusterDim.z = 1;
        at2[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at2[1].val.programmaticStreamSerializationAllowed = g.pdl ? 1 : 0;
        cfg2.attrs = at2;
        cfg2.numAttrs = 2;
        e = cudaLaunchKernelEx(&cfg2, pick_kernel_2sm(g.p.act, g.p.fmt, g.p.pk_nl > 0), g.p, n_items);
        count_launch();
        return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(workers * g.p.n_det);
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = g.smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = g.pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, k, g.p, n_items);
    count_launch();
    return e;
}

// ---------------------------------------------------------------------------------------------
// SIMT cross-check over the SAME operands and segment table (selected with gw_set_conv_impl; used by
// tests to tell "tensor-core plumbing bug" from "operand construction bug").  One thread per output.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float ld16v(const void* p, size_t i, int fmt) {
    if (fmt == FMT_BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[i]);
    return __half2float(reinterpret_cast<const __half*>(p)[i]);
}

__device__ float simt_dot(const ConvGemmParams& p, int batch, int det, int m, int n) {
    float acc = 0.f;
    const int row_off = p.a_count ? static_cast<int>((*p.a_count % p.a_ring_W) / p.a_ring_div) : 0;
    const size_t ktot = static_cast<size_t>(p.n_seg) * kSegK;
    for (int s = 0; s < p.n_seg; ++s) {
        const int r = m + p.seg_shift[s];
        if (r < 0 || r >= p.a_rows) continue;
        const size_t abase = (static_cast<size_t>(batch) * p.a_rows_tm + row_off + r) * p.a_cols + p.seg_col[s];
        const size_t bbase = (static_cast<size_t>(det) * p.N + n) * ktot + static_cast<size_t>(s) * kSegK;
        for (int k = 0; k < kSegK; ++k) acc = fmaf(ld16v(p.A, abase + k, p.fmt), ld16v(p.B, bbase + k, p.fmt), acc);
    }
    return acc;
}

__global__ void __launch_bounds__(128) k_conv_gemm_simt(const __grid_constant__ ConvGemmParams p) {
    const int batch = blockIdx.z;
    const int det = batch % p.n_det;
    const float* bias = p.bias + static_cast<size_t>(det) * p.N;
    if (p.epi == EPI_STORE) {
        const int n = blockIdx.x * blockDim.x + threadIdx.x;
        const int m = blockIdx.y;
        if (n >= p.N || m >= p.M) return;
        const float v = act_apply(simt_dot(p, batch, det, m, n) + bias[n], p.act);
        const size_t o = (static_cast<size_t>(batch) * p.M + m) * p.N + n;
        if (p.fmt == FMT_BF16) reinterpret_cast<__nv_bfloat16*>(p.out)[o] = __float2bfloat16_rn(v);
        else reinterpret_cast<__half*>(p.out)[o] = __float2half_rn(v);
    } else {
        const int half = p.N / 2, Mq = p.M / 2;
        const int c = blockIdx.x * blockDim.x + threadIdx.x;
        const int q = blockIdx.y;
        if (c >= half || q >= Mq) return;
        float best = 0.f;
        for (int i = 0; i < 4; ++i) {
            const int m = 2 * q + i / 2, n = (i % 2) * half + c;
            best = fmaxf(best, simt_dot(p, batch, det, m, n) + bias[n]);
        }
        const size_t o = (static_cast<size_t>(batch) * Mq + q) * half + c;
        if (p.epi == EPI_POOL) {
            if (p.fmt == FMT_BF16) reinterpret_cast<__nv_bfloat16*>(p.out)[o] = __float2bfloat16_rn(best);
            else reinterpret_cast<__half*>(p.out)[o] = __float2half_rn(best);
        } else {
            p.pooled_dbg[o] = best;
        }
    }
}

__global__ void __launch_bounds__(128) k_head_simt(const __grid_constant__ ConvGemmParams p) {
    __shared__ float gap_s[256];
    __shared__ float hid_s[256];
    const int batch = blockIdx.x;
    const int half = p.N / 2, Mq = p.M / 2;
    for (int c = threadIdx.x; c < half; c += blockDim.x) {
        float s = 0.f;
        for (int q = 0; q < Mq; ++q) s += p.pooled_dbg[(static_cast<size_t>(batch) * Mq + q) * half + c];
        gap_s[c] = s / static_cast<float>(Mq);
    }
    __syncthreads();
    for (int h = threadIdx.x; h < p.head_hidden; h += blockDim.x) {
        float s = p.hb1[h];
        for (int c = 0; c < half; ++c) s = fmaf(p.hw1[static_cast<size_t>(h) * half + c], gap_s[c], s);
        hid_s[h] = fmaxf(s, 0.f);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        float z = p.hb2[0];
        for (int h = 0; h < p.head_hidden; ++h) z = fmaf(p.hw2[h], hid_s[h], z);
        p.scores[batch] = 1.f / (1.f + __expf(-z));
    }
}

cudaError_t launch_conv_gemm_simt(const GemmLaunch& g, cudaStream_t st) {
    if (g.p.out_ring_div || g.p.v_tiles != g.p.tiles_m) return cudaErrorNotSupported;   // cross-check kernel: full windows only
    if (g.p.epi == EPI_STORE) {
        dim3 grid((g.p.N + 127) / 128, g.p.M, g.batch);
        k_conv_gemm_simt<<<grid, 128, 0, st>>>(g.p);
        count_launch();
    } else {
        dim3 grid((g.p.N / 2 + 127) / 128, g.p.M / 2, g.batch);
        k_conv_gemm_simt<<<grid, 128, 0, st>>>(g.p);
        count_launch();
        if (g.p.epi == EPI_POOL_HEAD) {
            k_head_simt<<<g.batch, 128, 0, st>>>(g.p);
            count_launch();
        }
    }
    return cudaGetLastError();
}

}  // namespace gw
