// gw_kernels.cu -- the bandwidth-bound and CUDA-core kernels of the hot path:
//   a1 snapshot append, (test) snapshot read-out, a2 window gather + convert,
//   a4' the final 1-output-channel ConvTranspose1d, a5 aggregation + normalise + subtract,
//   a6' the first (2-channel) classifier conv block.
// Step names a1..a7 are those of DESIGN.md "Steps on the hot path".
#include <stdio.h>

#include "gw_common.cuh"

namespace gw {

long long g_kernel_launches = 0;

__device__ __forceinline__ float ld16(const void* p, size_t i, int fmt) {
    if (fmt == FMT_BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[i]);
    return __half2float(reinterpret_cast<const __half*>(p)[i]);
}
__device__ __forceinline__ uint32_t pack16(float a, float b, int fmt) {
    if (fmt == FMT_BF16) {
        __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
        return *reinterpret_cast<uint32_t*>(&v);
    }
    __half2 v = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void unpack16x8(const uint4& q, float (&f)[8], int fmt) {
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (fmt == FMT_BF16) {
            float2 v = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&w[i]));
            f[2 * i] = v.x; f[2 * i + 1] = v.y;
        } else {
            float2 v = __half22float2(*reinterpret_cast<const __half2*>(&w[i]));
            f[2 * i] = v.x; f[2 * i + 1] = v.y;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a1  Snapshot append: ring[row][(count + i) mod W] = new[row][i], i < S; the last
// block to finish advances the device-resident sample counter, so a captured graph replays
// unchanged.  VEC = 4: 128-bit loads and stores (S, W multiples of 4 => count is too).
// ---------------------------------------------------------------------------------------------
template <int VEC>
__global__ void __launch_bounds__(256) k_append(float* __restrict__ ring, const float* __restrict__ src,
                                                long long* count, unsigned* ticket, int n_rows, int W, int S) {
    const long long cnt = *count;
    const int h = static_cast<int>(cnt % W);
    const int per_row = S / VEC;
    const long long total = static_cast<long long>(n_rows) * per_row;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int row = static_cast<int>(i / per_row);
        const int j = static_cast<int>(i % per_row) * VEC;
        int slot = h + j;
        if (slot >= W) slot -= W;                       // S <= W, so one wrap at most
        if (VEC == 4) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(src + static_cast<size_t>(row) * S + j));
            *reinterpret_cast<float4*>(ring + static_cast<size_t>(row) * W + slot) = v;
        } else {
            ring[static_cast<size_t>(row) * W + slot] = __ldg(src + static_cast<size_t>(row) * S + j);
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(ticket, 1u);
        if (t == gridDim.x - 1) {
            *count = cnt + S;
            *ticket = 0;
            __threadfence();
        }
    }
}

void launch_append(float* ring, const float* new_samples, long long* count, unsigned* ticket, int n_rows, int W,
                   int S, cudaStream_t st) {
    const bool vec = (S % 4 == 0) && (W % 4 == 0);
    const long long total = static_cast<long long>(n_rows) * (vec ? S / 4 : S);
    int blocks = static_cast<int>((total + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    if (vec) k_append<4><<<blocks, 256, 0, st>>>(ring, new_samples, count, ticket, n_rows, W, S);
    else k_append<1><<<blocks, 256, 0, st>>>(ring, new_samples, count, ticket, n_rows, W, S);
    ++g_kernel_launches;
}

bool is_append_kernel(const void* func) {
    return func == reinterpret_cast<const void*>(&k_append<4>) || func == reinterpret_cast<const void*>(&k_append<1>);
}

// Test hook: time-ordered read-out of the ring, out[row][n] = ring[row][(count + n) mod W].
__global__ void __launch_bounds__(256) k_snapshot(const float* __restrict__ ring, float* __restrict__ out,
                                                  const long long* count, int n_rows, int W) {
    const int h = static_cast<int>(*count % W);
    const long long total = static_cast<long long>(n_rows) * W;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int row = static_cast<int>(i / W);
        const int n = static_cast<int>(i % W);
        int slot = h + n;
        if (slot >= W) slot -= W;
        out[i] = ring[static_cast<size_t>(row) * W + slot];
    }
}

void launch_snapshot(const float* ring, float* out, const long long* count, int n_rows, int W, cudaStream_t st) {
    const long long total = static_cast<long long>(n_rows) * W;
    int blocks = static_cast<int>((total + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_snapshot<<<blocks, 256, 0, st>>>(ring, out, count, n_rows, W);
    ++g_kernel_launches;
}

// ---------------------------------------------------------------------------------------------
// a2  Window gather + convert: the time-ordered window of each detector's witness channels,
// rounded RN-even to the 16-bit storage type, channels-last [n*D][W][cpad] (channels >= n_wit are
// zero).  One block transposes a 32-channel x 128-position tile through shared memory: reads are
// contiguous along time (128 B per warp request), writes are 16-byte stores covering contiguous
// 64-byte rows.
// ---------------------------------------------------------------------------------------------
constexpr int kGatherPos = 128;

__global__ void __launch_bounds__(256) k_gather(const float* __restrict__ ring, void* __restrict__ xw,
                                                const long long* count, const int* __restrict__ rows_map,
                                                int channels, int n_det, int n_wit, int W, int cpad, int fmt) {
    __shared__ float tile[32][kGatherPos + 1];
    const int h = static_cast<int>(*count % W);
    const int sd = blockIdx.y;                       // stream * n_det + det
    const int s = sd / n_det, d = sd % n_det;
    const int cb = blockIdx.z * 32;                  // channel chunk
    const int n0 = blockIdx.x * kGatherPos;
    const int tid = threadIdx.x;
    {
        const int pos = tid % kGatherPos;            // 128 positions, 2 channel groups of 16
        const int cg = tid / kGatherPos;
        const int n = n0 + pos;
        int slot = h + n;
        if (slot >= W) slot -= W;
#pragma unroll 4
        for (int k = 0; k < 16; ++k) {
            const int c = cb + cg * 16 + k;
            float v = 0.f;
            if (c < n_wit && n < W) {
                const int row = s * channels + __ldg(rows_map + d * n_wit + c);
                v = __ldg(ring + static_cast<size_t>(row) * W + slot);
            }
            tile[cg * 16 + k][pos] = v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int pos = it * 64 + tid / 4;           // 64 positions per pass, 4 threads x 8 channels each
        const int c0 = (tid % 4) * 8;
        const int n = n0 + pos;
        if (n < W) {
            uint4 q;
            q.x = pack16(tile[c0 + 0][pos], tile[c0 + 1][pos], fmt);
            q.y = pack16(tile[c0 + 2][pos], tile[c0 + 3][pos], fmt);
            q.z = pack16(tile[c0 + 4][pos], tile[c0 + 5][pos], fmt);
            q.w = pack16(tile[c0 + 6][pos], tile[c0 + 7][pos], fmt);
            uint16_t* dst = reinterpret_cast<uint16_t*>(xw) + (static_cast<size_t>(sd) * W + n) * cpad + cb + c0;
            *reinterpret_cast<uint4*>(dst) = q;
        }
    }
}

void launch_gather(const float* ring, void* xw, const long long* count, const int* rows_map, int n_streams,
                   int channels, int n_det, int n_wit, int W, int cpad, int fmt, cudaStream_t st) {
    dim3 grid((W + kGatherPos - 1) / kGatherPos, n_streams * n_det, cpad / 32);
    k_gather<<<grid, 256, 0, st>>>(ring, xw, count, rows_map, channels, n_det, n_wit, W, cpad, fmt);
    ++g_kernel_launches;
}

// ---------------------------------------------------------------------------------------------
// a4' Final ConvTranspose1d (cout = 1, stride 2, pad = K/2, output_padding 1) on CUDA cores in
// fp32: 7 x cin weights are far too thin for a tensor-core tile.  D3 of DESIGN.md:
//   y[2q + r] = b + sum_ci sum_{j : (r + pad - j) even} w[ci][j] x[q + (r + pad - j)/2][ci].
// Each thread forms the K per-tap dot products t_j[l] of ONE input row l, the block exchanges them
// through shared memory, then each thread emits the two outputs of its row.
// x: [batch][L][cpad] 16-bit, wt: [n_det][K][cpad] fp32, pred: [batch][2L] fp32.
// ---------------------------------------------------------------------------------------------
constexpr int kFcThreads = 256;
constexpr int kFcHalo = 4;
constexpr int kFcMaxK = 9;

__global__ void __launch_bounds__(kFcThreads) k_final_convt(const void* __restrict__ x,
                                                            const float* __restrict__ wt,
                                                            const float* __restrict__ bias,
                                                            float* __restrict__ pred, int n_det, int L, int cpad,
                                                            int K, int pad, int fmt) {
    extern __shared__ float sm[];
    float* w_s = sm;                                  // [K][cpad]
    float* t_s = sm + K * cpad;                       // [K][kFcThreads]
    const int b = blockIdx.y;
    const int det = b % n_det;
    const int rows_out = kFcThreads - 2 * kFcHalo;
    const int q0 = blockIdx.x * rows_out;
    const int tid = threadIdx.x;
    for (int i = tid; i < K * cpad; i += kFcThreads) w_s[i] = __ldg(wt + static_cast<size_t>(det) * K * cpad + i);
    __syncthreads();
    const int l = q0 - kFcHalo + tid;
    float t[kFcMaxK];
#pragma unroll
    for (int j = 0; j < kFcMaxK; ++j) t[j] = 0.f;
    if (l >= 0 && l < L) {
        const uint4* row = reinterpret_cast<const uint4*>(reinterpret_cast<const uint16_t*>(x) +
                                                          (static_cast<size_t>(b) * L + l) * cpad);
        for (int c8 = 0; c8 < cpad / 8; ++c8) {
            float f[8];
            unpack16x8(__ldg(row + c8), f, fmt);
#pragma unroll
            for (int j = 0; j < kFcMaxK; ++j) {
                if (j < K) {
                    const float* wj = w_s + j * cpad + c8 * 8;
#pragma unroll
                    for (int e = 0; e < 8; ++e) t[j] = fmaf(wj[e], f[e], t[j]);
                }
            }
        }
    }
#pragma unroll
    for (int j = 0; j < kFcMaxK; ++j)
        if (j < K) t_s[j * kFcThreads + tid] = t[j];
    __syncthreads();
    if (tid >= kFcHalo && tid < kFcThreads - kFcHalo && l < L) {
        float y[2];
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            float acc = __ldg(bias + det);
            for (int j = 0; j < K; ++j) {
                const int e = r + pad - j;
                if ((e & 1) == 0) acc += t_s[j * kFcThreads + tid + e / 2];   // e/2 exact: e is even
            }
            y[r] = acc;
        }
        *reinterpret_cast<float2*>(pred + static_cast<size_t>(b) * 2 * L + 2 * l) = make_float2(y[0], y[1]);
    }
}

void launch_final_convt(const void* x, const float* wt, const float* bias, float* pred, int batch, int n_det,
                        int L, int cpad, int K, int pad, int fmt, cudaStream_t st) {
    const int rows_out = kFcThreads - 2 * kFcHalo;
    dim3 grid((L + rows_out - 1) / rows_out, batch);
    const size_t smem = static_cast<size_t>(K) * (cpad + kFcThreads) * sizeof(float);
    k_final_convt<<<grid, kFcThreads, smem, st>>>(x, wt, bias, pred, n_det, L, cpad, K, pad, fmt);
    ++g_kernel_launches;
}

// ---------------------------------------------------------------------------------------------
// a5  Aggregation + window normalisation + subtraction, one pass (D7 of DESIGN.md; north_star
// (3)).  Per window position n of (stream, detector): absolute index a = count - W + n, ring slot
// (count + n) mod W.
//   HANN_OLA:    acc[slot] = (n >= W - S ? 0 : acc[slot]) + hann[n] * p[n]       (first cover resets)
//                nhat = acc[slot] * inv_wsum[n];   cleaned = strain[slot] - nhat
//   LAST_STRIDE: the ring stores nhat itself: positions [W-S-delta, W-delta) take p[n];
//                newer positions are not covered yet (nhat = 0).
// Samples with a < 0 (before the stream started) are written as 0 and never touch the state.
// Algorithmic traffic: read p, acc, strain; write acc, cleaned  = 20 bytes per sample.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_aggregate(const AggParams a) {
    const long long cnt = *a.count;
    const int W = a.W, S = a.S;
    const int h = static_cast<int>(cnt % W);
    const int sd = blockIdx.y;
    const int s = sd / a.n_det, d = sd % a.n_det;
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= W) return;
    const long long abs_idx = cnt - W + n;
    int slot = h + n;
    if (slot >= W) slot -= W;
    const size_t wi = static_cast<size_t>(sd) * W;
    float nhat = 0.f, cleaned = 0.f;
    if (abs_idx >= 0) {
        const float p = __ldg(a.pred + wi + n);
        if (a.agg == 0) {
            const float prev = (n >= W - S) ? 0.f : a.acc[wi + slot];
            const float acc = fmaf(__ldg(a.hann + n), p, prev);
            a.acc[wi + slot] = acc;
            nhat = acc * __ldg(a.inv_wsum + n);
        } else {
            if (n >= W - a.delta) nhat = 0.f;
            else if (n >= W - S - a.delta) { nhat = p; a.acc[wi + slot] = p; }
            else nhat = a.acc[wi + slot];
        }
        const float strain = __ldg(a.ring + (static_cast<size_t>(s) * a.channels + __ldg(a.strain_rows + d)) * W + slot);
        cleaned = strain - nhat;
    }
    if (a.running_out) a.running_out[wi + n] = cleaned;
    if (a.nhat_out) a.nhat_out[wi + n] = nhat;
    if (a.final_out) {
        const int f0 = (a.agg == 0) ? 0 : W - S - a.delta;
        const int i = n - f0;
        if (i >= 0 && i < S) a.final_out[static_cast<size_t>(sd) * S + i] = cleaned;
    }
    if (a.clf_in) {
        const int i = n - (W - a.delta - a.Lb);
        if (i >= 0 && i < a.Lb) a.clf_in[static_cast<size_t>(sd) * a.Lb + i] = cleaned;
    }
}

void launch_aggregate(const AggParams& a, cudaStream_t st) {
    dim3 grid((a.W + 255) / 256, a.n_streams * a.n_det);
    k_aggregate<<<grid, 256, 0, st>>>(a);
    ++g_kernel_launches;
}

// ---------------------------------------------------------------------------------------------
// a6' First classifier block (cin = number of detectors, K = 8): conv + bias + ReLU + MaxPool(pool)
// on CUDA cores in fp32 (GEMM K would be 16: one MMA k-step, all epilogue).  One warp = 32 output
// channels of one pooled position; x reads are warp broadcasts, the 64-byte output row is contiguous.
// x: [batch][cin][L] fp32; w: [cout][cin][K] fp32 (already rounded to the storage type);
// out: [batch][L/pool][cpad] 16-bit channels-last, channels >= cout zero.
// ---------------------------------------------------------------------------------------------
constexpr int kC1Q = 64;          // pooled positions per block
constexpr int kC1MaxTaps = 32;    // cin * K held in registers per lane

__global__ void __launch_bounds__(256) k_bbh_conv1(const float* __restrict__ x, const float* __restrict__ w,
                                                   const float* __restrict__ bias, void* __restrict__ out,
                                                   int cin, int L, int cout, int cpad, int K, int pad_l,
                                                   int pool, int fmt) {
    extern __shared__ float xs[];                       // [cin][kC1Q * pool + K - 1] input tile with halo
    const int b = blockIdx.y;
    const int Lq = L / pool;
    const int q0 = blockIdx.x * kC1Q;
    const int span = kC1Q * pool + K - 1;
    const int l0 = q0 * pool - pad_l;                   // first input position of the tile
    for (int i = threadIdx.x; i < cin * span; i += blockDim.x) {
        const int ci = i / span, l = l0 + i % span;
        xs[i] = (l >= 0 && l < L) ? __ldg(x + (static_cast<size_t>(b) * cin + ci) * L + l) : 0.f;
    }
    const int lane = threadIdx.x % 32, wrp = threadIdx.x / 32;
    const int c = lane + blockIdx.z * 32;
    float wr[kC1MaxTaps];
#pragma unroll
    for (int i = 0; i < kC1MaxTaps; ++i) wr[i] = (c < cout && i < cin * K) ? __ldg(w + static_cast<size_t>(c) * cin * K + i) : 0.f;
    const float bc = c < cout ? __ldg(bias + c) : 0.f;
    int off[kC1MaxTaps];                                // tap t reads xs[off[t] + position]
#pragma unroll
    for (int t = 0; t < kC1MaxTaps; ++t) off[t] = (t / K) * span + t % K;
    const int n_taps = cin * K;
    __syncthreads();
    const int q_per_warp = kC1Q / 8;
    for (int qi = 0; qi < q_per_warp; ++qi) {
        const int ql = wrp * q_per_warp + qi;           // pooled position inside the tile
        const int q = q0 + ql;
        if (q >= Lq) break;
        float best = 0.f;                               // ReLU output is >= 0
        for (int i = 0; i < pool; ++i) {
            float acc = bc;
#pragma unroll
            for (int t = 0; t < kC1MaxTaps; ++t) {
                if (t < n_taps) acc = fmaf(wr[t], xs[off[t] + ql * pool + i], acc);   // warp-broadcast read
            }
            best = fmaxf(best, acc);
        }
        if (c >= cout) best = 0.f;
        const float other = __shfl_down_sync(0xffffffffu, best, 1);
        if ((lane & 1) == 0) {
            uint32_t* dst = reinterpret_cast<uint32_t*>(reinterpret_cast<uint16_t*>(out) +
                                                        (static_cast<size_t>(b) * Lq + q) * cpad + c);
            *dst = pack16(best, other, fmt);
        }
    }
}

void launch_bbh_conv1(const float* x, const float* w, const float* b, void* out, int batch, int n_det, int L,
                      int cout, int cpad, int K, int pad_l, int pool, int fmt, cudaStream_t st) {
    const int Lq = L / pool;
    dim3 grid((Lq + kC1Q - 1) / kC1Q, batch, cpad / 32);
    const size_t smem = static_cast<size_t>(n_det) * (kC1Q * pool + K - 1) * sizeof(float);
    k_bbh_conv1<<<grid, 256, smem, st>>>(x, w, b, out, n_det, L, cout, cpad, K, pad_l, pool, fmt);
    ++g_kernel_launches;
}

}  // namespace gw
