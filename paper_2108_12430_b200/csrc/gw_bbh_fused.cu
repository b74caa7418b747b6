// gw_bbh_fused.cu -- a6: the whole BBH classifier (BASELINE.json configs[2]: Conv1d 2->32->64->128, k 8,
// ReLU, MaxPool 4, global average pool, dense 128->64->1, sigmoid) as ONE kernel with ONE CTA PER WINDOW.  Every
// activation lives in shared memory (north_star (2): "activations stay in shared memory where a layer fits"); nothing
// but the 32 KiB input window, the weights (L2-resident constants) and one score per window touches global memory.
//
// All three conv blocks run on the tensor cores (tcgen05.mma, accumulators in TMEM):
//   block 1 (cin <= 2 -> 32, M = 4 conv positions per row)   A = an im2col tile built by the worker warps: row r holds the 11
//            input samples [4r-3, 4r+7] of each channel as a (hi, lo) pair of 16-bit values (x = hi + lo to ~2^-22, so the
//            fp32 input is NOT rounded to the storage type: D8's numerics are kept), pre-scaled by a power of two that
//            brings the window into fp16 range; B = the 8-tap filter as a Toeplitz matrix with N = 4 phases x 32 channels.
//            One row = one pooled position: max-pool is a max over four TMEM column groups IN the thread.
//   block 2 (32 -> 64)   A = block 1's pooled output stored as "quad rows" (row R = positions 4R..4R+3 x 32 channels =
//            two 128-byte swizzled blocks); for each of the 4 output phases q and each tap j the operand is a row-shifted,
//            32-byte-offset view of the same tile (descriptor arithmetic only), B = the plain [cout][tap][cin] weights.
//            Four accumulators (one per phase) per 128 quad rows; max-pool again in the thread.
//   block 3 (64 -> 128)  operands SWAPPED: A = weights (M = 128 output channels), B = block 2's output [position][64 ch]
//            row-shifted per tap (N = 256 positions), so a thread owns one output channel and all positions: max-pool,
//            ReLU and the global average pool are column arithmetic in registers.
// then the dense head and the sigmoid (fp32, CUDA cores).  Roles: warp 0 loads weights (bulk copies) and issues every MMA;
// the eight worker warps stage the window, build block 1's im2col tiles and drain its accumulators one tile apart, then
// drain blocks 2 and 3.  The MMAs of block 2's first tile are issued between block 1's last tiles (the tensor pipe idles
// through most of block 1).
// Shared memory is time-shared: [act1 | later taps 4-7 of block 3's weights] [im2col x 2 | later act2] [W2]
// [W1 + input staging | later taps 0-3 of block 3's weights].
#include <stdio.h>

#include "gw_common.cuh"
#include "gw_ptx.cuh"

namespace gw {

// Diagnostic builds (GW_TRACE=1): CTA 0 prints the SM-cycle stamps of its three roles' milestones.
#ifdef GW_TRACE
#define BF_TR_DECL long long bt_[24] = {0}; const long long bt0_ = clock64();
#define BF_TR(i) bt_[i] = clock64() - bt0_;
#define BF_TR_PRINT(name, n) if (blockIdx.x == 0 && lane == 0) { printf("[bbh_fused %s]", name); for (int i_ = 0; i_ < n; ++i_) printf(" %lld", bt_[i_]); printf("\n"); }
#else
#define BF_TR_DECL
#define BF_TR(i)
#define BF_TR_PRINT(name, n)
#endif

constexpr int kBfWorkers = 256;
constexpr int kBfThreads = 32 + kBfWorkers;
constexpr int kBfAct1Blk = 264 * 128;                 // [256 quad rows + 8 zero rows] of one 128-byte column block
constexpr int kBfAct1 = (8 + 264 + 264) * 128;        // 8 zero rows, block 0 (+8 zero rows), block 1 (+8 zero rows): 68608
constexpr int kBfImTile = 128 * 128;                  // one im2col tile: 128 rows x 64 16-bit values
constexpr int kBfAct2 = (8 + 256 + 8) * 128;          // [position][64 channels] with 8 zero rows on either side: 34816
constexpr int kBfOffIm = kBfAct1;                     // im2col double buffer (32 KiB), later act2
constexpr int kBfOffW2 = kBfOffIm + kBfAct2;          // 103424
constexpr int kBfOffD = kBfOffW2 + kBbhW2Bytes;       // 136192: W1 + staging, later W3 taps 0-3
constexpr int kBfRegD = 65536;
constexpr int kBfOffMisc = kBfOffD + kBfRegD;         // 201728
constexpr int kBfMisc = 4096;
constexpr int kBfSmem = 1024 + kBfOffMisc + kBfMisc;  // + alignment slack
constexpr int kBfXOff = 68;                           // staged window: sample l at index kBfXOff + l; 68 zeros before
constexpr int kBfXS = kBfXOff + 4096 + 12;            // (FIR history 63 + conv padding 3, rounded up), 12 after: per channel
constexpr int kBfYSpan = 528;                         // whitened samples of one tile (D12)
static_assert(kBfOffIm % 1024 == 0 && kBfOffW2 % 1024 == 0 && kBfOffD % 1024 == 0 && kBfOffMisc % 1024 == 0, "operand alignment");
static_assert(kBbhW1Bytes + (2 * kBfXS + 2 * kBfYSpan) * 4 <= kBfRegD, "staging must fit beside W1");

bool bbh_fused_supported(int L, int cin, int hidden) {
    return L >= 512 && L <= 4096 && L % 512 == 0 && cin >= 1 && cin <= 2 && hidden >= 1 && hidden <= 64;
}

template <int FMT>
__device__ __forceinline__ uint32_t bf_pack(float a, float b) {
    if (FMT == FMT_BF16) {
        __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
        return *reinterpret_cast<uint32_t*>(&v);
    }
    __half2 v = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}
// (a, b) -> the 16-bit pair nearest to it and the 16-bit pair nearest to what that rounding lost
template <int FMT>
__device__ __forceinline__ void bf_split(float a, float b, uint32_t& hi, uint32_t& lo) {
    if (FMT == FMT_BF16) {
        const __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
        const float2 f = __bfloat1622float2(h);
        hi = *reinterpret_cast<const uint32_t*>(&h);
        lo = bf_pack<FMT>(a - f.x, b - f.y);
    } else {
        const __half2 h = __floats2half2_rn(a, b);
        const float2 f = __half22float2(h);
        hi = *reinterpret_cast<const uint32_t*>(&h);
        lo = bf_pack<FMT>(a - f.x, b - f.y);
    }
}

// A read-only global load the compiler may not sink below later (volatile) barriers: the dense head's operands are
// requested long before they are needed, so that their latency runs under block 3.
__device__ __forceinline__ float bf_ldg_early(const float* q) {
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(q));
    return v;
}

template <int FMT>
__global__ void __launch_bounds__(kBfThreads, 1) k_bbh_fused(const __grid_constant__ BbhFusedParams p) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* act1 = smem;
    uint8_t* im = smem + kBfOffIm;                         // [2][kBfImTile]
    uint8_t* act2 = smem + kBfOffIm;
    uint8_t* w2s = smem + kBfOffW2;
    uint8_t* regd = smem + kBfOffD;
    uint8_t* w1s = regd;
    float* xf = reinterpret_cast<float*>(regd + kBbhW1Bytes);      // [2 channels][kBfXS] the input window, fp32
    float* ys = xf + 2 * kBfXS;                                    // [2 channels][kBfYSpan] whitened samples of a tile (D12)
    float* bias1 = reinterpret_cast<float*>(smem + kBfOffMisc);    // [32]
    float* bias2 = bias1 + 32;                                     // [64]
    float* bias3 = bias2 + 64;                                     // [128]
    float* gws = bias3 + 128;                                      // [2][64] whitening taps
    float* gap_part = gws + 128;                                   // [2][128]
    float* gap_s = gap_part + 256;                                 // [128] (unused: the head reads gap_part)
    float* hid_s = gap_s + 128;                                    // [64]
    float* red_s = hid_s + 64;                                     // [16]
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kBfOffMisc + 3584);
    uint64_t* w1bar = bars;            uint64_t* w2bar = bars + 1;
    uint64_t* w3abar = bars + 2;       uint64_t* w3bbar = bars + 3;
    uint64_t* im_full = bars + 4;      uint64_t* im_empty = bars + 6;        // [2] each
    uint64_t* acc1_full = bars + 8;    uint64_t* acc1_empty = bars + 10;     // [2] each
    uint64_t* act1_done = bars + 12;                                         // [8], single use
    uint64_t* acc2_full = bars + 20;                                         // [2], single use
    uint64_t* p2_done = bars + 22;     uint64_t* act2_done = bars + 23;
    uint64_t* acc3_full = bars + 24;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 32);

    stamp_begin(p.stamp);
    BF_TR_DECL
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x / 32, 0);
    const int lane = threadIdx.x % 32;
    const int L = p.L;
    const int T1 = L / 512;                  // block-1 tiles: 128 pooled positions (512 conv positions) each
    const int T2 = (L / 16 + 127) / 128;     // block-2 tiles: 128 quad rows (512 block-2 conv positions) each
    const int P2 = L / 16;                   // block 2's pooled positions = block 3's conv positions
    const int P3 = L / 64;                   // block 3's pooled positions

    if (warp == 0) {
        if (lane == 0) {
            for (int i = 0; i < 4; ++i) mbar_init(&bars[i], 1);
            for (int i = 0; i < 2; ++i) {
                mbar_init(&im_full[i], 8); mbar_init(&im_empty[i], 1);
                mbar_init(&acc1_full[i], 1); mbar_init(&acc1_empty[i], 8);
                mbar_init(&acc2_full[i], 1);
            }
            for (int i = 0; i < 8; ++i) mbar_init(&act1_done[i], 8);
            mbar_init(p2_done, 1); mbar_init(act2_done, 8 * T2); mbar_init(acc3_full, 1);
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc(tmem_slot, 512);
    } else {
        // act1's zeros: the 8-row halos around both column blocks are the conv's zero padding, and the rows past the
        // window's last quad row are never written
        const int wt = threadIdx.x - 32;
        const int R1 = L / 16;
        for (int i = wt; i < (8 + 264 + 264) * 8; i += kBfWorkers) {
            const int r = i >> 3;
            const bool live = (r >= 8 && r < 8 + R1) || (r >= 272 && r < 272 + R1);
            if (!live) reinterpret_cast<uint4*>(act1)[i] = make_uint4(0, 0, 0, 0);
        }
        if (wt < 32) bias1[wt] = __ldg(p.b1 + wt);
        else if (wt < 96) bias2[wt - 32] = __ldg(p.b2 + wt - 32);
        else if (wt < 224) bias3[wt - 96] = __ldg(p.b3 + wt - 96);
        if (p.whiten && wt < 128) gws[wt] = (wt / 64 < p.cin && wt % 64 < p.whiten_n) ? __ldg(p.whiten + (wt / 64) * p.whiten_n + wt % 64) : 0.f;
        fence_proxy_async();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);
    griddep_launch_dependents();

    if (warp == 0) {
        // ------------------------------------------------------------ weight loads + every MMA of the three blocks
        if (lane == 0) {                                   // constants of the engine: nothing the predecessor writes
            mbar_arrive_expect_tx(w1bar, kBbhW1Bytes);
            bulk_load_1d(w1s, p.w1img, kBbhW1Bytes, w1bar);
            mbar_arrive_expect_tx(w2bar, kBbhW2Bytes);
            for (int i = 0; i < 2; ++i) bulk_load_1d(w2s + i * 16384, p.w2img + i * 16384, 16384, w2bar);
        }
        __syncwarp();
        const uint32_t leader = elect_one() ? 1u : 0u;
        const uint32_t idesc1 = umma_idesc_f16(FMT, kTileM, 128);
        const uint32_t idesc2 = umma_idesc_f16(FMT, kTileM, 64);
        const uint32_t idesc3 = umma_idesc_f16(FMT, kTileM, 256);
        BF_TR(0)
        mbar_wait(w1bar, 0);
        BF_TR(1)
        // block 1: D[r][q*32 + co] = sum_k im2col[r][k] . W1[q*32 + co][k], four K steps (channel x (hi | lo))
        // block 2: output phase q of quad row R, tap j reads pooled-1 position 4R + q + j - 3 = quad row R + sh, slot qq;
        //          one chunk = the 16 MMAs of one phase.  The tensor pipe idles through most of block 1 (an im2col tile is
        //          4 MMAs), so the chunks of block 2's first tile are issued BETWEEN block 1's last tiles, as soon as the
        //          block-1 tiles that tile reads (0 .. need0) have been drained.
        const uint32_t w1_lo = umma_desc_lo(smem_u32(w1s));
        const uint32_t act1_u32 = smem_u32(act1) + 1024, w2_u32 = smem_u32(w2s);
        int done = 0;                                      // act1_done barriers waited for so far
        auto chunk = [&](int t2, int q) {
            const uint32_t d_tmem = tmem_base + (t2 == 0 ? 256u : 0u) + q * 64;   // tile 0 beside block 1's stages, tile 1 over them
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int v = q + j + 1;                   // q + j - 3 + 4
                const int sh = v / 4 - 1, qq = v % 4;
                const uint32_t a_lo = umma_desc_lo(act1_u32 + (qq >> 1) * kBfAct1Blk + (128 * t2 + sh) * 128 + (qq & 1) * 64);
                const uint32_t b_lo = umma_desc_lo(w2_u32 + (j >> 1) * 8192 + (j & 1) * 64);
#pragma unroll
                for (int k = 0; k < 2; ++k)
                    umma_f16_if(leader, d_tmem, umma_desc_make(a_lo + 2 * k), umma_desc_make(b_lo + 2 * k), idesc2, (j | k) ? 1u : 0u);
            }
        };
        const int need0 = min(4, T1 - 1);                  // last block-1 tile that block 2's first tile reads (its halo row)
        int q_next = 0;
        for (int t = 0; t < T1; ++t) {
            const int s = t & 1;
            const uint32_t ph = (t >> 1) & 1;
            mbar_wait(&acc1_empty[s], ph ^ 1);
            mbar_wait(&im_full[s], ph);
            if (t == 0) { BF_TR(2) }
            tc_fence_after();
            const uint32_t a_lo = umma_desc_lo(smem_u32(im + s * kBfImTile));
#pragma unroll
            for (int k = 0; k < 4; ++k)
                umma_f16_if(leader, tmem_base + s * 128, umma_desc_make(a_lo + 2 * k), umma_desc_make(w1_lo + 2 * k), idesc1, k ? 1u : 0u);
            umma_commit_if(leader, &im_empty[s]);
            umma_commit_if(leader, &acc1_full[s]);
            if (t > need0 && q_next < 4) {
                if (q_next == 0) {
                    mbar_wait(w2bar, 0);
                    while (done <= need0) { mbar_wait(&act1_done[done], 0); ++done; }
                    tc_fence_after();
                    BF_TR(4)
                }
                chunk(0, q_next++);
            }
        }
        BF_TR(3)
        if (q_next == 0) {
            mbar_wait(w2bar, 0);
            while (done <= need0) { mbar_wait(&act1_done[done], 0); ++done; }
            tc_fence_after();
            BF_TR(4)
        }
        while (q_next < 4) chunk(0, q_next++);
        umma_commit_if(leader, &acc2_full[0]);
        while (done < T1) { mbar_wait(&act1_done[done], 0); ++done; }
        tc_fence_after();
        BF_TR(5)
        // block 1 is over: W1 and the input staging are dead, the first four taps of block 3 take their place
        if (lane == 0) {
            fence_proxy_async();
            mbar_arrive_expect_tx(w3abar, 4 * 16384);
            for (int i = 0; i < 4; ++i) bulk_load_1d(regd + i * 16384, p.w3img + i * 16384, 16384, w3abar);
        }
        __syncwarp();
        if (T2 == 2) {
            for (int q = 0; q < 4; ++q) chunk(1, q);
            umma_commit_if(leader, &acc2_full[1]);
        }
        // act1 is dead once block 2's MMAs have retired: taps 4-7 of block 3 take its place
        BF_TR(6)
        umma_commit_if(leader, p2_done);
        mbar_wait(p2_done, 0);
        BF_TR(7)
        if (lane == 0) {
            fence_proxy_async();
            mbar_arrive_expect_tx(w3bbar, 4 * 16384);
            for (int i = 0; i < 4; ++i) bulk_load_1d(act1 + i * 16384, p.w3img + (4 + i) * 16384, 16384, w3bbar);
        }
        __syncwarp();
        // block 3, operands swapped: D[co][pos] = sum_{j, ci} W3[co][j][ci] . act2[pos + j - 3][ci]
        mbar_wait(act2_done, 0);
        BF_TR(8)
        mbar_wait(w3abar, 0);
        BF_TR(9)
        tc_fence_after();
        const uint32_t act2_u32 = smem_u32(act2);
        for (int j = 0; j < 8; ++j) {
            if (j == 4) { BF_TR(10) mbar_wait(w3bbar, 0); tc_fence_after(); }
            const uint32_t a_lo = umma_desc_lo(j < 4 ? smem_u32(regd) + j * 16384 : smem_u32(act1) + (j - 4) * 16384);
            const uint32_t b_lo = umma_desc_lo(act2_u32 + (8 + j - 3) * 128);
#pragma unroll
            for (int k = 0; k < 4; ++k)
                umma_f16_if(leader, tmem_base + 256, umma_desc_make(a_lo + 2 * k), umma_desc_make(b_lo + 2 * k), idesc3, (j | k) ? 1u : 0u);
        }
        umma_commit_if(leader, acc3_full);
        BF_TR(11)
        BF_TR_PRINT("mma: w-issued w1 im0 p1-issued act1(t2=0) act1(t2=1) p2-issued p2-retired act2 w3a j4 p3-issued", 12)
    } else {
        const int wt = threadIdx.x - 32;                   // 0..255
        const int ww = warp - 1;                           // 0..7
        const int quad = warp % 4;                         // the TMEM lane quadrant this warp may read
        const uint32_t lane_base = static_cast<uint32_t>(quad * 32) << 16;
        const float* xb = p.x + static_cast<size_t>(blockIdx.x) * p.cin * L;
        const int half = ww / 4;                           // which half of a tile's channels this warp drains
        griddep_wait();                                    // the window is the predecessor's output
        BF_TR(0)
        // ---- the whole window into shared memory (fp32, zeros on either side: the conv's padding and the FIR's zero
        // initial state) and, on the way, max|x| for the power-of-two scale: |x| (after whitening: <= max|x| * sum|g|) < s,
        // so that the (hi, lo) pair of a sample is in fp16 range whatever units the strain comes in
        float amax = 0.f;
        const int L4 = L / 4;
        float4 xv[8];                                      // cin * L / 4 <= 2048 float4 = 8 per thread
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int i = wt + e * kBfWorkers;
            xv[e] = i < p.cin * L4 ? __ldg(reinterpret_cast<const float4*>(xb) + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            amax = fmaxf(amax, fmaxf(fmaxf(fabsf(xv[e].x), fabsf(xv[e].y)), fmaxf(fabsf(xv[e].z), fabsf(xv[e].w))));
        }
        for (int i = wt; i < 2 * (kBfXOff + 12); i += kBfWorkers) {
            const int ch = i / (kBfXOff + 12), k = i % (kBfXOff + 12);
            xf[ch * kBfXS + (k < kBfXOff ? k : L + k)] = 0.f;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        if (lane == 0) red_s[ww] = amax;
        asm volatile("bar.sync 1, 256;" ::: "memory");
        amax = red_s[0];
#pragma unroll
        for (int i = 1; i < 8; ++i) amax = fmaxf(amax, red_s[i]);
        if (p.whiten) {
            float gsum = 0.f;
            for (int ch = 0; ch < p.cin; ++ch) {
                float s = 0.f;
                for (int j = 0; j < p.whiten_n; ++j) s += fabsf(gws[ch * 64 + j]);
                gsum = fmaxf(gsum, s);
            }
            amax *= gsum;
        }
        float scale = 1.f, inv_scale = 1.f;
        {
            const uint32_t E = (__float_as_uint(amax) >> 23) & 0xffu;
            if (E >= 1 && E <= 252) { scale = __uint_as_float((E + 1) << 23); inv_scale = __uint_as_float((253 - E) << 23); }
        }
        // the staged window is x / s (exact: a power of two); whitening is linear, block 1's epilogue multiplies by s
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const int i = wt + e * kBfWorkers;
            if (i < p.cin * L4) {
                const int ch = i >= L4 ? 1 : 0;
                *reinterpret_cast<float4*>(xf + ch * kBfXS + kBfXOff + 4 * (i - ch * L4)) =
                    make_float4(xv[e].x * inv_scale, xv[e].y * inv_scale, xv[e].z * inv_scale, xv[e].w * inv_scale);
            }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        BF_TR(1)

        // ---------------------------------------------------------------------------------- block 1
        // Every warp does both jobs, one tile apart: build (one (row, channel) of the im2col tile per thread), then drain
        // the previous tile's accumulators (max over the 4 phases, bias, ReLU -> act1).
        for (int t = 0; t <= T1; ++t) {
            if (t < T1) {
                const int buf = t & 1;
                const int b = wt & 127, ch = wt >> 7;      // row in the tile (pooled position 128 t + b), input channel
                const float* src = xf + ch * kBfXS + kBfXOff - 4 + 512 * t;      // src[i]: sample 512 t - 4 + i
                if (p.whiten) {
                    // D12: y[l] = sum_j g[j] x[l - j], zero initial state at the window start; outside [0, L) the conv's padding
                    asm volatile("bar.sync 1, 256;" ::: "memory");               // the previous tile's rows have been built
                    for (int idx = wt; idx < p.cin * 520; idx += kBfWorkers) {
                        const int c = idx >= 520 ? 1 : 0, i = idx - c * 520;
                        const int l = 512 * t - 4 + i;
                        float v = 0.f;
                        if (l >= 0 && l < L) {
                            const float* xs = xf + c * kBfXS + kBfXOff + l;
                            for (int j = 0; j < p.whiten_n; ++j) v = fmaf(gws[c * 64 + j], xs[-j], v);
                        }
                        ys[c * kBfYSpan + i] = v;
                    }
                    asm volatile("bar.sync 1, 256;" ::: "memory");
                    src = ys + ch * kBfYSpan;
                }
                float v[12];
                if (ch < p.cin) {
                    const float4* s4 = reinterpret_cast<const float4*>(src + 4 * b);
#pragma unroll
                    for (int i = 0; i < 3; ++i) {
                        const float4 f = s4[i];
                        v[4 * i] = f.x; v[4 * i + 1] = f.y; v[4 * i + 2] = f.z; v[4 * i + 3] = f.w;
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < 12; ++i) v[i] = 0.f;
                }
                // e_i = v[1 + i], i = 0..10: sample 4 (128 t + b) - 3 + i
                uint32_t hi[8], lo[8];
#pragma unroll
                for (int i = 0; i < 5; ++i) bf_split<FMT>(v[1 + 2 * i], v[2 + 2 * i], hi[i], lo[i]);
                bf_split<FMT>(v[11], 0.f, hi[5], lo[5]);
                hi[6] = hi[7] = lo[6] = lo[7] = 0u;
                if (t == 3) { BF_TR(12) }
                mbar_wait(&im_empty[buf], ((t >> 1) & 1) ^ 1);
                if (t == 3) { BF_TR(13) }
                const uint32_t row_u32 = smem_u32(im + buf * kBfImTile) + b * 128;
                const int c0 = ch * 4;                     // 16-byte chunks: (channel, part) x 2
                sts_u4(row_u32 + (((c0 + 0) ^ (b & 7)) << 4), hi[0], hi[1], hi[2], hi[3]);
                sts_u4(row_u32 + (((c0 + 1) ^ (b & 7)) << 4), hi[4], hi[5], hi[6], hi[7]);
                sts_u4(row_u32 + (((c0 + 2) ^ (b & 7)) << 4), lo[0], lo[1], lo[2], lo[3]);
                sts_u4(row_u32 + (((c0 + 3) ^ (b & 7)) << 4), lo[4], lo[5], lo[6], lo[7]);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&im_full[buf]);
                if (t == 0) { BF_TR(2) }
                if (t == 3) { BF_TR(14) }
            }
            if (t > 0) {
                const int te = t - 1, s = te & 1;
                const int b = quad * 32 + lane;
                mbar_wait(&acc1_full[s], (te >> 1) & 1);
                if (t == 3) { BF_TR(15) }
                tc_fence_after();
                const uint32_t taddr = tmem_base + lane_base + s * 128 + half * 16;
                uint32_t r0[16], r1[16], r2[16], r3[16];
                tmem_ld_32x16(taddr, r0);
                tmem_ld_32x16(taddr + 32, r1);
                tmem_ld_32x16(taddr + 64, r2);
                tmem_ld_32x16(taddr + 96, r3);
                tmem_ld_wait();
                if (t == 3) { BF_TR(16) }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc1_empty[s]);
                uint32_t out[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float m0 = fmaxf(fmaxf(__uint_as_float(r0[2 * i]), __uint_as_float(r1[2 * i])), fmaxf(__uint_as_float(r2[2 * i]), __uint_as_float(r3[2 * i])));
                    const float m1 = fmaxf(fmaxf(__uint_as_float(r0[2 * i + 1]), __uint_as_float(r1[2 * i + 1])), fmaxf(__uint_as_float(r2[2 * i + 1]), __uint_as_float(r3[2 * i + 1])));
                    out[i] = bf_pack<FMT>(fmaxf(fmaf(m0, scale, bias1[half * 16 + 2 * i]), 0.f), fmaxf(fmaf(m1, scale, bias1[half * 16 + 2 * i + 1]), 0.f));
                }
                const int P = 128 * te + b, R = P >> 2, u = P & 3;
                const uint32_t row_u32 = smem_u32(act1) + 1024 + (u >> 1) * kBfAct1Blk + R * 128;
                const int c0 = (u & 1) * 4 + half * 2;
                sts_u4(row_u32 + (((c0 + 0) ^ (R & 7)) << 4), out[0], out[1], out[2], out[3]);
                sts_u4(row_u32 + (((c0 + 1) ^ (R & 7)) << 4), out[4], out[5], out[6], out[7]);
                if (t == 3) { BF_TR(17) }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&act1_done[te]);
                if (te == 0) { BF_TR(3) }
                if (t == 3) { BF_TR(18) }
            }
        }

        // ---------------------------------------------------- block 2, epilogue (all eight warps) -> act2 [position][64]
        // block 2: this warp drains channels [32 half, +32) of its lane quadrant
        mbar_wait(&acc2_full[0], 0);                       // every block-1 MMA has retired: the im2col tiles are dead
        BF_TR(4)
        if (wt < 128) {
            // rows nobody writes: the 8-row halos and everything past the last tile (zero padding of block 3)
            const int first = 8 + 128 * T2, n_tail = (8 + 256 + 8) - first;
            for (int i = wt; i < (8 + n_tail) * 8; i += 128) {
                const int r = i / 8 < 8 ? i / 8 : first + i / 8 - 8;
                *reinterpret_cast<uint4*>(act2 + r * 128 + (i % 8) * 16) = make_uint4(0, 0, 0, 0);
            }
        }
        for (int t2 = 0; t2 < T2; ++t2) {
            if (t2) mbar_wait(&acc2_full[t2], 0);
            tc_fence_after();
            const uint32_t taddr = tmem_base + lane_base + (t2 == 0 ? 256u : 0u) + half * 32;
            const int row = 128 * t2 + quad * 32 + lane;
            uint32_t out[16];
#pragma unroll
            for (int hc = 0; hc < 2; ++hc) {
                uint32_t r0[16], r1[16], r2[16], r3[16];
                tmem_ld_32x16(taddr + hc * 16, r0);
                tmem_ld_32x16(taddr + 64 + hc * 16, r1);
                tmem_ld_32x16(taddr + 128 + hc * 16, r2);
                tmem_ld_32x16(taddr + 192 + hc * 16, r3);
                tmem_ld_wait();
                float o[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float m = fmaxf(fmaxf(__uint_as_float(r0[i]), __uint_as_float(r1[i])), fmaxf(__uint_as_float(r2[i]), __uint_as_float(r3[i])));
                    o[i] = fmaxf(m + bias2[half * 32 + hc * 16 + i], 0.f);
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) out[hc * 8 + i] = row < P2 ? bf_pack<FMT>(o[2 * i], o[2 * i + 1]) : 0u;
            }
            const uint32_t row_u32 = smem_u32(act2) + 1024 + row * 128;
#pragma unroll
            for (int c4 = 0; c4 < 4; ++c4)
                sts_u4(row_u32 + (((half * 4 + c4) ^ (row & 7)) << 4), out[4 * c4], out[4 * c4 + 1], out[4 * c4 + 2], out[4 * c4 + 3]);
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(act2_done);
            if (t2 == 0) { BF_TR(5) } else { BF_TR(6) }
        }

        // ---------------------------- block 3, epilogue: a thread owns channel co; pool, ReLU and the average are in registers
        // everything the dense head reads from global memory is requested BEFORE the wait for block 3's accumulators: this
        // warp's rows of the first dense layer (hidden <= 64: 8 rows x 4 values per lane), their biases, the second layer
        float wreg[8][4], hb1v[8];
#pragma unroll
        for (int rr = 0; rr < 8; ++rr) {
            const int hrow = ww + rr * 8;
            const int hr = hrow < p.hidden ? hrow : 0;     // rows past `hidden` are loaded (row 0) and never used
            hb1v[rr] = bf_ldg_early(p.hb1 + hr);
#pragma unroll
            for (int k = 0; k < 4; ++k) wreg[rr][k] = bf_ldg_early(p.hw1 + static_cast<size_t>(hr) * 128 + lane + 32 * k);
        }
        const float hw2a = bf_ldg_early(p.hw2 + (lane < p.hidden ? lane : 0)), hw2b = bf_ldg_early(p.hw2 + (lane + 32 < p.hidden ? lane + 32 : 0));
        const float hb2v = bf_ldg_early(p.hb2);
        mbar_wait(acc3_full, 0);
        BF_TR(7)
        tc_fence_after();
        {
            const int co = quad * 32 + lane;
            const float bc = bias3[co];
            float sum = 0.f;
#pragma unroll
            for (int ch = 0; ch < 4; ch += 2) {
                uint32_t ra[32], rb[32];
                tmem_ld_32x32(tmem_base + lane_base + 256 + half * 128 + ch * 32, ra);
                tmem_ld_32x32(tmem_base + lane_base + 256 + half * 128 + ch * 32 + 32, rb);
                tmem_ld_wait();
#pragma unroll
                for (int g = 0; g < 16; ++g) {
                    const uint32_t* r = g < 8 ? ra : rb;
                    const int gg = g & 7;
                    const float m = fmaxf(fmaxf(__uint_as_float(r[4 * gg]), __uint_as_float(r[4 * gg + 1])),
                                          fmaxf(__uint_as_float(r[4 * gg + 2]), __uint_as_float(r[4 * gg + 3])));
                    if (half * 32 + ch * 8 + g < P3) sum += fmaxf(m + bc, 0.f);
                }
            }
            gap_part[half * 128 + co] = sum;
        }
        BF_TR(19)
        asm volatile("bar.sync 1, 256;" ::: "memory");
        BF_TR(20)
        // dense 128 -> hidden + ReLU (one warp per hidden unit, lanes over the inputs), dense hidden -> 1, sigmoid
        {
            const float inv_p3 = 1.f / static_cast<float>(P3);
            float gv[4], sr[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) gv[k] = (gap_part[lane + 32 * k] + gap_part[128 + lane + 32 * k]) * inv_p3;
#pragma unroll
            for (int rr = 0; rr < 8; ++rr) {
                sr[rr] = 0.f;
#pragma unroll
                for (int k = 0; k < 4; ++k) sr[rr] = fmaf(wreg[rr][k], gv[k], sr[rr]);
            }
            // the eight butterflies in lockstep (row by row they would be eight serial chains of five shuffles)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int rr = 0; rr < 8; ++rr) sr[rr] += __shfl_xor_sync(0xffffffffu, sr[rr], o);
            if (lane < 8 && ww + lane * 8 < p.hidden) {
                float mine = sr[0], bm = hb1v[0];
#pragma unroll
                for (int rr = 1; rr < 8; ++rr) if (lane == rr) { mine = sr[rr]; bm = hb1v[rr]; }
                hid_s[ww + lane * 8] = fmaxf(mine + bm, 0.f);
            }
        }
        BF_TR(21)
        asm volatile("bar.sync 1, 256;" ::: "memory");
        BF_TR(22)
        if (wt < 32) {
            float s = 0.f;
            if (lane < p.hidden) s = fmaf(hw2a, hid_s[lane], s);
            if (lane + 32 < p.hidden) s = fmaf(hw2b, hid_s[lane + 32], s);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (wt == 0) p.scores[blockIdx.x] = 1.f / (1.f + __expf(-(s + hb2v)));
        }
        BF_TR(8)
        if (ww == 0) { BF_TR_PRINT("worker: wait scale im[0] act1[0] acc2[0] act2[0] act2[1] acc3 end - - - | t3: built im_empty arrived acc1_full tmem_ld stored arrived | gap bar dense bar", 23) }
    }
    tc_fence_before();
    __syncthreads();
    stamp_end(p.stamp);
    if (warp == 0) tmem_dealloc(tmem_base, 512);
}

static bool g_bf_prepared = false;
cudaError_t bbh_fused_prepare() {
    if (g_bf_prepared) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_bbh_fused<FMT_FP16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBfSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_bbh_fused<FMT_BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBfSmem);
    g_bf_prepared = e == cudaSuccess;
    return e;
}

cudaError_t launch_bbh_fused(const BbhFusedParams& p, int batch, int fmt, int pdl, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(batch);
    cfg.blockDim = dim3(kBfThreads);
    cfg.dynamicSmemBytes = kBfSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = fmt == FMT_BF16 ? cudaLaunchKernelEx(&cfg, k_bbh_fused<FMT_BF16>, p)
                                          : cudaLaunchKernelEx(&cfg, k_bbh_fused<FMT_FP16>, p);
    count_launch();
    return e;
}

}  // namespace gw
