// gwstream: the one entry point that allocates nothing (include/gwstream.h, gw_ola_offline_noalloc).
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
// the offline periodic-Hann overlap-add of per-window predictions (D9), the kernel
// k_ola_offline of gw_kernels.cu, with the scratch that kernel needs -- the Hann window and the summed window weights along
// every residue chain, which gw_offline_create keeps in cudaMalloc'ed tables -- in a file-scope __device__ array of fixed size.
// Every GPU that loads the library holds those kOlaScratchBytes until the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: the address comes from cudaGetSymbolAddress,
// once per device with that device current (ola_scratch_for_current_device below), and is what the kernels are given.
// All calls on a device share the array and it keeps the last call's contents.  Nothing in it has to start at zero: the two
// set-up kernels of a call rewrite every entry (n < window) that its overlap-add kernel reads, stream-ordered before it.
// Calls that overlap on the GPU (two streams, or two threads on one device) race on the tables unless they use the same
// (window, stride); calls on one stream are ordered.
#include <math.h>
#include <stdio.h>

#include <mutex>

#include "../../include/gwstream.h"
#include "gw_common.cuh"

namespace gw {

constexpr int kOlaMaxWindow = GW_OLA_NOALLOC_MAX_WINDOW;                 // 32768 samples = the paper's 8 s window at 4096 Hz
constexpr size_t kOlaOffW64 = 0;                                          // double w[n]   = 0.5 - 0.5 cos(2 pi n / W)
constexpr size_t kOlaOffCum = static_cast<size_t>(kOlaMaxWindow) * 8;     // double cum[n] = sum_{i >= 0, n + iS < W} w[n + iS]
constexpr size_t kOlaOffHann = static_cast<size_t>(kOlaMaxWindow) * 16;   // float  hann[n] = (float) w[n]
constexpr size_t kOlaScratchBytes = static_cast<size_t>(kOlaMaxWindow) * 20;   // 640 KiB

static __device__ __align__(256) unsigned char g_ola_scratch[kOlaScratchBytes];

// Set-up 1: the periodic Hann window in double (the expression and operation order of the host tables in gw_engine.cu)
// and rounded to float.
__global__ void __launch_bounds__(256) k_ola_noalloc_window(unsigned char* __restrict__ scratch, int W) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= W) return;
    const double pi = 3.14159265358979323846;
    const double w = 0.5 - 0.5 * cos(2.0 * pi * n / W);
    reinterpret_cast<double*>(scratch + kOlaOffW64)[n] = w;
    reinterpret_cast<float*>(scratch + kOlaOffHann)[n] = static_cast<float>(w);
}

// Set-up 2: summed weights along the residue chain that starts at n, added in ascending order (the streaming path's table).
__global__ void __launch_bounds__(256) k_ola_noalloc_chain(unsigned char* __restrict__ scratch, int W, int S) {
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= W) return;
    const double* w = reinterpret_cast<const double*>(scratch + kOlaOffW64);
    double sum = 0.0;
    for (int m = n; m < W; m += S) sum += w[m];
    reinterpret_cast<double*>(scratch + kOlaOffCum)[n] = sum;
}

// The overlap-add itself: k_ola_offline's arithmetic (same fused multiply-add chain over the covering windows in ascending
// order, same normaliser), with the strain rows passed directly ([D][T]) and the tables read from the scratch array.
__global__ void __launch_bounds__(256) k_ola_noalloc(const float* __restrict__ pred, const float* __restrict__ strain,
                                                     const unsigned char* __restrict__ scratch, float* __restrict__ cleaned,
                                                     float* __restrict__ nhat_out, const float* __restrict__ post, int B,
                                                     int n_det, int W, int S, long long T) {
    const long long a = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
    const int d = blockIdx.y;
    if (a >= T) return;
    const float* hann = reinterpret_cast<const float*>(scratch + kOlaOffHann);
    const double* cum = reinterpret_cast<const double*>(scratch + kOlaOffCum);
    const int k = W / S;
    const int q = static_cast<int>(a / S), r = static_cast<int>(a % S);
    const int j_lo = q - k + 1 > 0 ? q - k + 1 : 0;
    const int j_hi = q < B - 1 ? q : B - 1;
    float acc = 0.f;
    for (int j = j_lo; j <= j_hi; ++j) {
        const int n = static_cast<int>(a - static_cast<long long>(j) * S);
        acc = fmaf(hann[n], __ldg(pred + (static_cast<size_t>(j) * n_det + d) * W + n), acc);
    }
    const int n_new = r + (q - j_hi) * S;                  // position in the newest covering window
    const int n_past = r + (q - j_lo + 1) * S;             // first position of the chain NOT covered
    const double sum = cum[n_new] - (n_past < W ? cum[n_past] : 0.0);
    const float ps = post ? __ldg(post + 2 * d) : 1.f, pm = post ? __ldg(post + 2 * d + 1) : 0.f;
    const float nhat = sum > 0.0 ? fmaf(ps, acc * static_cast<float>(1.0 / sum), pm) : 0.f;
    cleaned[static_cast<size_t>(d) * T + a] = __ldg(strain + static_cast<size_t>(d) * T + a) - nhat;
    if (nhat_out) nhat_out[static_cast<size_t>(d) * T + a] = nhat;
}

// Device address of the scratch array on the CURRENT device; looked up once per device, under a lock, no allocation.
constexpr int kOlaMaxDevices = 64;
static std::mutex g_ola_mu;
static unsigned char* g_ola_ptr[kOlaMaxDevices];

static cudaError_t ola_scratch_for_current_device(unsigned char** out, int* dev_out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= kOlaMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_ola_mu);
    if (!g_ola_ptr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_ola_scratch);
        if (e != cudaSuccess) return e;
        g_ola_ptr[dev] = static_cast<unsigned char*>(ptr);
    }
    *out = g_ola_ptr[dev];
    return cudaSuccess;
}

}  // namespace gw

using namespace gw;

extern "C" int gw_ola_offline_noalloc(const float* pred_dev, const float* strain_dev, float* cleaned_dev, float* noise_dev,
                                      const float* post_dev, int n_windows, int n_det, int window, int stride, void* stream) {
    char msg[256];
    if (!pred_dev || !strain_dev || !cleaned_dev) return report_error(GW_EINVAL, "gw_ola_offline_noalloc: NULL argument");
    if (n_windows < 1 || n_det < 1 || n_det > 65535 || window < 1 || stride < 1)
        return report_error(GW_EINVAL, "gw_ola_offline_noalloc: bad shape");
    if (window % stride != 0 || window / stride < 2)
        return report_error(GW_EINVAL, "gw_ola_offline_noalloc: overlap-add needs window % stride == 0 and window/stride >= 2");
    if (window > kOlaMaxWindow) {
        snprintf(msg, sizeof msg, "gw_ola_offline_noalloc: window %d exceeds the built-in scratch (GW_OLA_NOALLOC_MAX_WINDOW = %d samples); "
                 "use gw_offline_create / gw_offline_run", window, kOlaMaxWindow);
        return report_error(GW_EINVAL, msg);
    }
    const long long T = static_cast<long long>(window) + static_cast<long long>(n_windows - 1) * stride;
    if ((T + 255) / 256 > 2147483647LL) return report_error(GW_EINVAL, "gw_ola_offline_noalloc: segment too long for one launch");
    unsigned char* scratch = nullptr;
    int dev = -1;
    cudaError_t e = ola_scratch_for_current_device(&scratch, &dev);
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "gw_ola_offline_noalloc: scratch address on device %d: %s (gwstream has no CPU fallback)", dev,
                 cudaGetErrorString(e));
        return report_error(GW_ECUDA, msg);
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const unsigned wblocks = static_cast<unsigned>((window + 255) / 256);
    k_ola_noalloc_window<<<wblocks, 256, 0, st>>>(scratch, window);
    count_launch();
    k_ola_noalloc_chain<<<wblocks, 256, 0, st>>>(scratch, window, stride);
    count_launch();
    dim3 grid(static_cast<unsigned>((T + 255) / 256), static_cast<unsigned>(n_det));
    k_ola_noalloc<<<grid, 256, 0, st>>>(pred_dev, strain_dev, scratch, cleaned_dev, noise_dev, post_dev, n_windows, n_det, window,
                                        stride, T);
    count_launch();
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        snprintf(msg, sizeof msg, "gw_ola_offline_noalloc: launch: %s", cudaGetErrorString(e));
        return report_error(GW_ECUDA, msg);
    }
    return GW_OK;
}
