// gw_conv_gemm.cu -- every Conv1d / ConvTranspose1d layer with enough channels as an implicit GEMM on
// the 5th-generation tensor cores (tcgen05.mma, accumulator in TMEM, operands staged by TMA).
//
//   D[m][n] = sum_s  A[m + shift_s][col_s .. col_s + 64) . B[n][64 s .. 64 s + 64)
//
// A is a 2-D view of the channels-last input activation of one (stream, detector):
//   stride-2 Conv1d (encoder):   rows = L/2 position pairs, cols = 2 Cin (even | odd position)
//   stride-2 ConvTranspose1d:    rows = L positions,        cols = Cin; N = (even | odd output) x Cout
//   stride-1 Conv1d + pool 4:    rows = L/2 position pairs, cols = 2 Cin; N = (even | odd output) x Cout
// so every tap is a row-shifted rectangular tile that one TMA box load fetches, and the layer's zero
// padding is TMA's out-of-bounds fill (the batch index is the third tensor dimension, so a shifted
// tile never bleeds into the neighbouring window).  B is the per-detector weight matrix, K-major,
// built on the host at create time.
//
// Warp roles (192 threads): warp 0 = TMA producer (+ TMEM alloc/dealloc), warp 1 = MMA issuer (one
// thread), warps 2..5 = epilogue (TMEM -> registers -> bias/activation/pool -> 16-bit global).
#include <stdio.h>

#include "gw_common.cuh"
#include "gw_ptx.cuh"

namespace gw {

constexpr int kGemmThreads = 192;
constexpr int kABytes = kTileM * 128;   // 128 rows x 128 bytes

int conv_gemm_smem_bytes(int N, int stages) { return stages * (kABytes + N * 128) + 1024 /*align*/ + 256 /*barriers*/; }

__device__ __forceinline__ float act_apply(float v, int act) {
    if (act == ACT_TANH) {
        // tanh(v) = 1 - 2/(1 + e^{2v}): two MUFU ops (ex2, rcp), absolute error ~1e-7.  The one-op
        // tanh.approx.f32 (relative error 2^-11) is as large as a bf16 rounding step and 4x an fp16 one,
        // and it flips ~10% of the storage roundings; the epilogue is not the bottleneck.
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

__global__ void __launch_bounds__(kGemmThreads, 1) k_conv_gemm_umma(const __grid_constant__ ConvGemmParams p,
                                                                    int stages) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int b_bytes = p.N * 128;
    const int stage_bytes = kABytes + b_bytes;
    uint64_t* full_bar = reinterpret_cast<uint64_t*>(smem + stages * stage_bytes);
    uint64_t* empty_bar = full_bar + stages;
    uint64_t* tmem_full_bar = empty_bar + stages;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tmem_full_bar + 1);

    const int warp = threadIdx.x / 32;
    const int lane = threadIdx.x % 32;
    const int m0 = blockIdx.x * kTileM;
    const int batch = blockIdx.y;
    const int det = batch % p.n_det;

    uint32_t tmem_cols = 32;
    while (tmem_cols < static_cast<uint32_t>(p.N)) tmem_cols <<= 1;

    if (warp == 0) {
        if (lane == 0) {
            tma_prefetch_desc(&p.tmA);
            tma_prefetch_desc(&p.tmB);
            for (int i = 0; i < stages; ++i) {
                mbar_init(&full_bar[i], 1);
                mbar_init(&empty_bar[i], 1);
            }
            mbar_init(tmem_full_bar, 1);
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc(tmem_slot, tmem_cols);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        if (lane == 0) {
            for (int s = 0; s < p.n_seg; ++s) {
                const int stage = s % stages;
                const uint32_t phase = (s / stages) & 1;
                mbar_wait(&empty_bar[stage], phase ^ 1);
                mbar_arrive_expect_tx(&full_bar[stage], stage_bytes);
                uint8_t* a_dst = smem + stage * stage_bytes;
                tma_load_3d(a_dst, &p.tmA, &full_bar[stage], p.seg_col[s], m0 + p.seg_shift[s], batch);
                tma_load_3d(a_dst + kABytes, &p.tmB, &full_bar[stage], s * kSegK, 0, det);
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            const uint32_t idesc = umma_idesc_f16(p.fmt, kTileM, p.N);
            for (int s = 0; s < p.n_seg; ++s) {
                const int stage = s % stages;
                const uint32_t phase = (s / stages) & 1;
                mbar_wait(&full_bar[stage], phase);
                tc_fence_after();
                const uint32_t a_addr = smem_u32(smem + stage * stage_bytes);
                const uint64_t adesc = umma_smem_desc_sw128(a_addr);
                const uint64_t bdesc = umma_smem_desc_sw128(a_addr + kABytes);
#pragma unroll
                for (int k = 0; k < kSegK / 16; ++k) {
                    // advance 16 elements = 32 bytes along K inside the 128-byte swizzle row: +2 in the
                    // (addr >> 4) field of the descriptor
                    umma_f16(tmem_base, adesc + 2 * k, bdesc + 2 * k, idesc, (s | k) != 0 ? 1u : 0u);
                }
                umma_commit(&empty_bar[stage]);        // frees the smem slot when these MMAs retire
            }
            umma_commit(tmem_full_bar);                // accumulator complete
        }
    } else {
        // ------------------------------------------------------------------ epilogue warps 2..5
        const int quad = warp % 4;                     // TMEM lane quadrant this warp may read
        const int row_in_tile = quad * 32 + lane;
        const int row = m0 + row_in_tile;
        mbar_wait(tmem_full_bar, 0);
        tc_fence_after();
        const uint32_t taddr = tmem_base + (static_cast<uint32_t>(quad * 32) << 16);
        const float* bias = p.bias + static_cast<size_t>(det) * p.N;
        if (p.epi == EPI_STORE) {
            uint16_t* orow = reinterpret_cast<uint16_t*>(p.out) + (static_cast<size_t>(batch) * p.M + row) * p.N;
            for (int c0 = 0; c0 < p.N; c0 += 32) {
                uint32_t r[32];
                tmem_ld_32x32(taddr + c0, r);
                tmem_ld_wait();
                if (row < p.M) {
                    uint32_t o[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const float v0 = act_apply(__uint_as_float(r[2 * j]) + __ldg(bias + c0 + 2 * j), p.act);
                        const float v1 = act_apply(__uint_as_float(r[2 * j + 1]) + __ldg(bias + c0 + 2 * j + 1), p.act);
                        o[j] = pack_pair(v0, v1, p.fmt);
                    }
                    uint4* dst = reinterpret_cast<uint4*>(orow + c0);
#pragma unroll
                    for (int j = 0; j < 4; ++j) dst[j] = make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
                }
            }
        } else {
            // conv (stride 1) + bias + ReLU + MaxPool(4): row m holds outputs 2m (cols [0,N/2)) and 2m+1
            // (cols [N/2,N)); pooled row q = m/2 is the max over both halves of rows 2q and 2q+1.
            const int half = p.N / 2;
            const int Mq = p.M / 2;
            float* pool_s = reinterpret_cast<float*>(smem);             // [64][half+1] fp32, pipeline smem is free now
            const int pstride = half + 1;
            for (int c0 = 0; c0 < half; c0 += 32) {
                uint32_t re[32], ro[32];
                tmem_ld_32x32(taddr + c0, re);
                tmem_ld_32x32(taddr + half + c0, ro);
                tmem_ld_wait();
                float v[32];
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    const float bj = __ldg(bias + c0 + j);
                    float m = fmaxf(__uint_as_float(re[j]) + bj, __uint_as_float(ro[j]) + bj);
                    m = (row < p.M) ? fmaxf(m, 0.f) : 0.f;               // ReLU; rows past the end contribute 0
                    const float other = __shfl_xor_sync(0xffffffffu, m, 1);
                    v[j] = fmaxf(m, other);
                }
                if ((lane & 1) == 0 && row < p.M) {
                    const int q = row / 2;
                    if (p.epi == EPI_POOL) {
                        uint16_t* orow = reinterpret_cast<uint16_t*>(p.out) + (static_cast<size_t>(batch) * Mq + q) * half + c0;
                        uint4* dst = reinterpret_cast<uint4*>(orow);
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            dst[j] = make_uint4(pack_pair(v[8 * j], v[8 * j + 1], p.fmt), pack_pair(v[8 * j + 2], v[8 * j + 3], p.fmt),
                                                pack_pair(v[8 * j + 4], v[8 * j + 5], p.fmt), pack_pair(v[8 * j + 6], v[8 * j + 7], p.fmt));
                    } else {
                        float* prow = pool_s + (row_in_tile / 2) * pstride + c0;
#pragma unroll
                        for (int j = 0; j < 32; ++j) prow[j] = v[j];
                    }
                }
            }
            if (p.epi == EPI_POOL_HEAD) {
                // global average pool over the Mq pooled rows, dense(half -> hidden) + ReLU,
                // dense(hidden -> 1), sigmoid: fused into this (last) conv block's epilogue.
                float* gap_s = pool_s + 64 * pstride;                    // [half]
                float* hid_s = gap_s + half;                             // [hidden]
                const int et = threadIdx.x - 64;                         // 0..127 among the epilogue threads
                asm volatile("bar.sync 1, 128;" ::: "memory");
                for (int c = et; c < half; c += 128) {
                    float s = 0.f;
                    for (int q = 0; q < Mq; ++q) s += pool_s[q * pstride + c];
                    gap_s[c] = s / static_cast<float>(Mq);
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
                for (int hrow = et; hrow < p.head_hidden; hrow += 128) {
                    float s = __ldg(p.hb1 + hrow);
                    const float* wr = p.hw1 + static_cast<size_t>(hrow) * half;
                    for (int c = 0; c < half; ++c) s = fmaf(__ldg(wr + c), gap_s[c], s);
                    hid_s[hrow] = fmaxf(s, 0.f);
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
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
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, tmem_cols);
}

static bool g_prepared = false;
cudaError_t conv_gemm_prepare() {
    if (g_prepared) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_conv_gemm_umma, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e == cudaSuccess) g_prepared = true;
    return e;
}

void launch_conv_gemm_umma(const GemmLaunch& g, cudaStream_t st) {
    dim3 grid((g.p.M + kTileM - 1) / kTileM, g.batch);
    k_conv_gemm_umma<<<grid, kGemmThreads, g.smem_bytes, st>>>(g.p, g.stages);
    ++g_kernel_launches;
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
    const size_t ktot = static_cast<size_t>(p.n_seg) * kSegK;
    for (int s = 0; s < p.n_seg; ++s) {
        const int r = m + p.seg_shift[s];
        if (r < 0 || r >= p.a_rows) continue;
        const size_t abase = (static_cast<size_t>(batch) * p.a_rows + r) * p.a_cols + p.seg_col[s];
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

void launch_conv_gemm_simt(const GemmLaunch& g, cudaStream_t st) {
    if (g.p.epi == EPI_STORE) {
        dim3 grid((g.p.N + 127) / 128, g.p.M, g.batch);
        k_conv_gemm_simt<<<grid, 128, 0, st>>>(g.p);
        ++g_kernel_launches;
    } else {
        dim3 grid((g.p.N / 2 + 127) / 128, g.p.M / 2, g.batch);
        k_conv_gemm_simt<<<grid, 128, 0, st>>>(g.p);
        ++g_kernel_launches;
        if (g.p.epi == EPI_POOL_HEAD) {
            k_head_simt<<<g.batch, 128, 0, st>>>(g.p);
            ++g_kernel_launches;
        }
    }
}

}  // namespace gw
