// gw_engine.cu -- host side of libgwstream: the C ABI of include/gwstream.h, parameter preparation
// (BatchNorm fold, rounding to the storage type, GEMM operand construction), TMA descriptors, the
// per-update launch sequence and its CUDA-graph capture.  No arithmetic of the per-update path runs on
// the host; everything here is one-time setup or launch plumbing.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <string>
#include <vector>

#include "../../include/gwstream.h"
#include "../../include/gwstream_diag.h"
#include "gw_common.cuh"

using namespace gw;

// ------------------------------------------------------------------------------------ errors
// Every handle starts with a HandleBase: gw_last_error(handle) finds the handle's own message there.  fail() records
// the message for the calling thread (create failures return no handle) and for the handle the running call is on.
static constexpr uint32_t kHandleMagic = 0x47577331u;   // "GWs1"
struct HandleBase {
    uint32_t magic = kHandleMagic;
    std::string err;
};
static thread_local std::string g_err;
static thread_local HandleBase* g_cur = nullptr;         // handle of the API call running on this thread
struct CallScope {
    HandleBase* prev;
    explicit CallScope(const void* h) : prev(g_cur) { g_cur = const_cast<HandleBase*>(static_cast<const HandleBase*>(h)); }
    ~CallScope() { g_cur = prev; }
};

static int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    if (g_cur && g_cur->magic == kHandleMagic) g_cur->err = buf;
    return code;
}
// fail() for the library's other translation units (gw_noalloc.cu): a finished message, no formatting
int gw::report_error(int code, const char* msg) { return fail(code, "%s", msg); }
#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t _e = (expr);                                                                  \
        if (_e != cudaSuccess)                                                                    \
            return fail(_e == cudaErrorMemoryAllocation ? GW_ENOMEM : GW_ECUDA, "%s: %s", #expr,  \
                        cudaGetErrorString(_e));                                                  \
    } while (0)

extern "C" const char* gw_last_error(const void* handle) {
    if (handle) {
        const HandleBase* b = static_cast<const HandleBase*>(handle);
        if (b->magic == kHandleMagic) return b->err.c_str();
    }
    return g_err.c_str();
}
extern "C" int64_t gw_kernel_launches(void) { return kernel_launches(); }

extern "C" void gw_options_default(gw_options* o) {
    if (!o) return;
    o->conv_impl = GW_IMPL_UMMA;
    o->fuse_tail = 1; o->pdl = 1; o->snake = 1; o->two_sm = 1; o->skip_zeros = 1;
    o->incremental = 0;
    o->fuse_bbh = 1;
    o->fuse_head = 1;
}
static int take_options(gw_options& dst, const gw_options* src) {
    gw_options_default(&dst);
    if (!src) return GW_OK;
    if (src->conv_impl != GW_IMPL_UMMA && src->conv_impl != GW_IMPL_SIMT) return fail(GW_EINVAL, "unknown conv impl %d", src->conv_impl);
    dst = *src;
    dst.fuse_tail = !!src->fuse_tail; dst.pdl = !!src->pdl; dst.snake = !!src->snake; dst.two_sm = !!src->two_sm;
    dst.skip_zeros = !!src->skip_zeros; dst.incremental = !!src->incremental; dst.fuse_bbh = !!src->fuse_bbh; dst.fuse_head = !!src->fuse_head;
    return GW_OK;
}

static int check_device() {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) return fail(GW_ECUDA, "no CUDA device (%s); gwstream has no CPU fallback",
                                                cudaGetErrorString(e));
    return GW_OK;
}

extern "C" int gw_probe_mma_cycles(int N, float* issue_cycles, float* complete_cycles) {
    if (!issue_cycles || !complete_cycles) return fail(GW_EINVAL, "gw_probe_mma_cycles: NULL argument");
    if (N != 16 && N != 32 && N != 64 && N != 128 && N != 256) return fail(GW_EINVAL, "gw_probe_mma_cycles: N must be 16, 32, 64, 128 or 256");
    if (int rc = check_device()) return rc;
    CU_TRY(probe_mma_cycles(N, issue_cycles, complete_cycles));
    return GW_OK;
}

extern "C" int gw_probe_mufu_rate(int mode, int threads, float* results_per_clock_per_sm) {
    if (!results_per_clock_per_sm) return fail(GW_EINVAL, "gw_probe_mufu_rate: NULL argument");
    if (mode < 0 || mode > 2) return fail(GW_EINVAL, "gw_probe_mufu_rate: mode must be 0 (tanh.f32), 1 (tanh.f16x2) or 2 (ex2 + rcp)");
    if (threads < 32 || threads > 1024 || threads % 32) return fail(GW_EINVAL, "gw_probe_mufu_rate: threads must be a multiple of 32 in [32, 1024]");
    if (int rc = check_device()) return rc;
    CU_TRY(probe_mufu_rate(mode, threads, results_per_clock_per_sm));
    return GW_OK;
}

// ------------------------------------------------------------------------- TMA descriptor encode
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static PFN_encodeTiled g_encode = nullptr;

static int get_encode() {
    if (g_encode) return GW_OK;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || fn == nullptr || qres != cudaDriverEntryPointSuccess)
        return fail(GW_ECUDA, "cuTensorMapEncodeTiled not available: %s", cudaGetErrorString(e));
    g_encode = reinterpret_cast<PFN_encodeTiled>(fn);
    return GW_OK;
}

// 4-D tensor of 16-bit elements (offline first layer: cols, rows, detector, window), box (64, box1, 1, 1), 128B swizzle.
static int make_tmap4(CUtensorMap* tm, const void* base, int fmt, uint64_t d0, uint64_t d1, uint64_t d2, uint64_t d3,
                      uint64_t stride1, uint64_t stride2, uint64_t stride3, uint32_t box1) {
    if (int rc = get_encode()) return rc;
    cuuint64_t dims[4] = {d0, d1, d2, d3};
    cuuint64_t strides[3] = {stride1 * 2, stride2 * 2, stride3 * 2};
    cuuint32_t box[4] = {kSegK, box1, 1, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = g_encode(tm, fmt == FMT_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 4,
                          const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(GW_ECUDA, "cuTensorMapEncodeTiled (4-D) failed (%d)", (int)r);
    return GW_OK;
}

// 3-D tensor of 16-bit elements, dims (d0 fastest, d1, d2), strides in elements, box (64, box1, 1), 128B swizzle.
static int make_tmap(CUtensorMap* tm, const void* base, int fmt, uint64_t d0, uint64_t d1, uint64_t d2,
                     uint64_t stride1, uint64_t stride2, uint32_t box1, uint32_t box0 = kSegK) {
    if (int rc = get_encode()) return rc;
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {stride1 * 2, stride2 * 2};
    cuuint32_t box[3] = {box0, box1, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    // the swizzle span equals the box row: 64 elements = 128 bytes, 32 elements = 64 bytes
    const CUtensorMapSwizzle sw = box0 * 2 == 128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
    CUresult r = g_encode(tm, fmt == FMT_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3,
                          const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                          sw, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(GW_ECUDA, "cuTensorMapEncodeTiled failed (%d) dims %llu,%llu,%llu", (int)r,
                                       (unsigned long long)d0, (unsigned long long)d1, (unsigned long long)d2);
    return GW_OK;
}

// --------------------------------------------------------------------- storage-type rounding (host)
// Round a double straight to the 16-bit storage grid, nearest-even, and return the 16-bit pattern.
// p = significand bits incl. the hidden one, emin = smallest normal exponent.
static uint16_t to_storage_bits(double v, int fmt) {
    const int p = fmt == FMT_BF16 ? 8 : 11;
    const int emin = fmt == FMT_BF16 ? -126 : -14;
    float f;
    if (v == 0.0 || !isfinite(v)) {
        f = static_cast<float>(v);
    } else {
        int e = ilogb(v);
        if (e < emin) e = emin;
        const int sh = e - (p - 1);                   // exponent of one unit in the last place
        const double q = scalbn(v, -sh);              // exact
        double fl = floor(q);
        const double diff = q - fl;
        if (diff > 0.5 || (diff == 0.5 && fmod(fl, 2.0) != 0.0)) fl += 1.0;
        f = static_cast<float>(scalbn(fl, sh));       // exactly representable in float
    }
    if (fmt == FMT_BF16) {
        uint32_t u;
        memcpy(&u, &f, 4);
        return static_cast<uint16_t>(u >> 16);        // low 16 bits are zero by construction
    }
    __half h = __float2half_rn(f);                    // exact: f is on the fp16 grid (or overflows to inf)
    uint16_t b;
    memcpy(&b, &h, 2);
    return b;
}
static double storage_to_double(uint16_t b, int fmt) {
    if (fmt == FMT_BF16) {
        uint32_t u = static_cast<uint32_t>(b) << 16;
        float f;
        memcpy(&f, &u, 4);
        return f;
    }
    __half h;
    memcpy(&h, &b, 2);
    return __half2float(h);
}

// ------------------------------------------------------------------------------ folded host layer
struct HostLayer {
    int kind, cin, cout, k, stride, pad_l, pad_r, act, pool;
    std::vector<double> w, b;                        // BatchNorm folded, double
    double W(int o, int i, int j) const {            // weight connecting input channel i to output channel o, tap j
        return kind == GW_CONV ? w[(static_cast<size_t>(o) * cin + i) * k + j] : w[(static_cast<size_t>(i) * cout + o) * k + j];
    }
};

static int fold_layer(const gw_conv_layer& L, HostLayer& H) {
    if (L.cin < 1 || L.cout < 1 || L.k < 1 || L.k > 9 || !L.w || !L.b) return fail(GW_EINVAL, "bad conv layer");
    H.kind = L.kind; H.cin = L.cin; H.cout = L.cout; H.k = L.k; H.stride = L.stride;
    H.pad_l = L.pad_l; H.pad_r = L.pad_r; H.act = L.act; H.pool = L.pool < 1 ? 1 : L.pool;
    const size_t nw = static_cast<size_t>(L.cin) * L.cout * L.k;
    H.w.resize(nw); H.b.resize(L.cout);
    for (size_t i = 0; i < nw; ++i) H.w[i] = L.w[i];
    for (int c = 0; c < L.cout; ++c) H.b[c] = L.b[c];
    if (L.bn_gamma) {
        if (!L.bn_beta || !L.bn_mean || !L.bn_var) return fail(GW_EINVAL, "incomplete BatchNorm parameters");
        for (int co = 0; co < L.cout; ++co) {
            const double g = static_cast<double>(L.bn_gamma[co]) / sqrt(static_cast<double>(L.bn_var[co]) + static_cast<double>(L.bn_eps));
            for (int ci = 0; ci < L.cin; ++ci)
                for (int j = 0; j < L.k; ++j) {
                    const size_t idx = L.kind == GW_CONV ? (static_cast<size_t>(co) * L.cin + ci) * L.k + j
                                                         : (static_cast<size_t>(ci) * L.cout + co) * L.k + j;
                    H.w[idx] *= g;
                }
            H.b[co] = (H.b[co] - static_cast<double>(L.bn_mean[co])) * g + static_cast<double>(L.bn_beta[co]);
        }
    }
    return GW_OK;
}

static int round_up(int v, int m) { return (v + m - 1) / m * m; }

// ------------------------------------------------------------------------------ launch context
// What every enqueue helper needs: the stream, the first CUDA error of the sequence (launch errors are sticky and
// reported by the API call), and -- only while the PROFILING graph is captured -- the device array of %globaltimer
// stamps plus the host-side list of kernel labels in launch order (gw_step_profile).
constexpr int kMaxStamps = 32;
struct Prof {
    std::vector<std::string> labels;
    std::vector<double> flops, smem;               // executed algorithmic FLOPs / shared-memory bytes per kernel
};
struct LaunchCtx {
    cudaStream_t st = nullptr;
    unsigned long long* stamps = nullptr;          // device [kMaxStamps][kStampSlots] or null
    Prof* prof = nullptr;
    cudaError_t err = cudaSuccess;
    explicit LaunchCtx(cudaStream_t s) : st(s) {}
    Stamp next(const std::string& label, double flops = 0.0, double smem = 0.0) {
        if (!stamps || !prof) return nullptr;
        const int i = static_cast<int>(prof->labels.size());
        if (i >= kMaxStamps) return nullptr;
        prof->labels.push_back(label); prof->flops.push_back(flops); prof->smem.push_back(smem);
        return stamps + kStampSlots * i;
    }
    void check(cudaError_t e) { if (err == cudaSuccess && e != cudaSuccess) err = e; }
};
#define CX_TRY(cx, what)                                                                                   \
    do {                                                                                                   \
        if ((cx).err != cudaSuccess) return fail(GW_ECUDA, "%s: %s", what, cudaGetErrorString((cx).err));  \
    } while (0)

// ------------------------------------------------------------------------------------ handles
struct gw_stream {
    HandleBase base;
    int n, C, fs, W, S;
    float* ring = nullptr;
    long long* d_count = nullptr;
    unsigned* d_ticket = nullptr;
    int64_t updates = 0;
    gw_deepclean* dc = nullptr;
};

enum GemmKind { GK_ENC, GK_DEC, GK_BBH };

struct GemmLayer {
    GemmLaunch g;                                // whole windows
    GemmLaunch gi;                               // incremental path: the two recomputed zones only (when has_inc)
    bool has_inc = false;
    void* d_B = nullptr;
    float* d_bias = nullptr;
    CUtensorMap* d_heads = nullptr;              // incremental path, CTA-pair layers: one input tensor map per window head
    CUtensorMap* d_heads_left = nullptr;         // the same with a box of pk_nl rows (zones packed into one tile)
    CUtensorMap* d_heads_right = nullptr;        // ... and of pk_nr rows
    int impl = GW_IMPL_UMMA;
    std::string name;                            // profiler label, e.g. "gemm.dc3"
    double flops = 0.0;                          // algorithmic FLOPs per batch item, whole window (real channels and taps only)
};

struct gw_deepclean {
    HandleBase base;
    gw_options opt;
    gw_stream* s = nullptr;
    int n_det = 0, n_layers = 0, n_wit = 0, agg = 0, delta = 0, fmt = FMT_BF16;
    int batch = 0;
    std::vector<HostLayer> host;                 // [n_det * n_layers]
    std::vector<GemmLayer> gemm;                 // layers 0 .. n_layers-2
    void* ring16 = nullptr;                      // mirror ring [batch][2W][cpad0], 16-bit (when `mirror`)
    bool offline = false;                        // owned by a gw_offline: windows of one archival segment
    long long off_T = 0;                         // offline: samples per channel of the segment
    void* seg16 = nullptr;                       // offline: 16-bit channels-last segment [n_det][T][cpad0]; the first layer
                                                 // reads its overlapping windows straight from it (null: gather path)
    bool mirror = false;                         // first layer reads the window from ring16 (no per-update gather)
    bool fused_tail = false;                     // last GEMM layer + final ConvTranspose1d run as one kernel (EPI_FINAL)
    bool inc = false;                            // incremental path: act[i] are mirror rings [batch][2 L_i][C_i], pred a ring
    bool has_chain = false;                      // gw_options.fuse_head: layers 0 and 1 run as ONE kernel (EPI_CHAIN); act[1] is
    GemmLayer chain;                             // never written.  Operands are those of gemm[0] / gemm[1] (not owned here)
    std::vector<void*> act;                      // act[0] = gathered window (null when `mirror`), act[i+1] = output of layer i
    std::vector<int> act_rows, act_cols;
    float* d_wt_final = nullptr;                 // [n_det][K][cpad]
    float* d_b_final = nullptr;                  // [n_det]
    void* d_fin_B = nullptr;                     // fused tail: last layer as a 16-bit B operand [n_det][16][3 x 64]
    int final_K = 0, final_pad = 0, final_cpad = 0, final_L = 0;
    float* pred = nullptr;                       // [batch][W]
    float* acc = nullptr;                        // [batch][W]
    float* nhat = nullptr;                       // [batch][W] (test hook, allocated lazily)
    float* d_hann = nullptr;
    float* d_inv_wsum = nullptr;
    int* d_rows_map = nullptr;
    int* d_strain_rows = nullptr;
    float* d_pre = nullptr;                      // [n_det][n_wit][2] witness standardisation (mean, 1/std); identity (0, 1)
    float* d_post = nullptr;                     // [n_det][2] estimate back to strain units (std, mean); identity (1, 0)
    float* final_buf = nullptr;                  // [batch][S]
    float* d_fir = nullptr;                      // D11: post-filter taps [fir_n] (null: off)
    float* d_hist = nullptr;                     // D11: [2][batch][kMaxFir - 1] emitted samples carried between updates
    int fir_n = 0;
    float* clf_in = nullptr;                     // owned by the attached gw_bbh
    int Lb = 0;
    gw_bbh* bbh = nullptr;
    int64_t forward_for = 0, cleaned_for = 0;
};

struct gw_bbh {
    HandleBase base;
    gw_options opt;
    gw_deepclean* dc = nullptr;
    int n_det = 0, batch = 0, fmt = FMT_BF16, L = 0;
    HostLayer c1;
    float* d_w1 = nullptr;                       // first conv, fp32 (rounded to the storage grid)
    float* d_b1 = nullptr;
    int c1_cpad = 0;
    std::vector<GemmLayer> gemm;
    std::vector<void*> act;
    float* in_buf = nullptr;                     // [batch][n_det][L]
    float *d_hw1 = nullptr, *d_hb1 = nullptr, *d_hw2 = nullptr, *d_hb2 = nullptr;
    float* pooled_dbg = nullptr;
    float* scores_buf = nullptr;
    float* d_whiten = nullptr;                   // D12: whitening taps [n_det][whiten_n] (null: off)
    int whiten_n = 0;
    int64_t scored_for = 0;
    // gw_options.fuse_bbh: the whole classifier as one shared-memory-resident kernel (gw_bbh_fused.cu)
    bool fused = false;
    uint8_t *d_w1img = nullptr, *d_w2img = nullptr, *d_w3img = nullptr;
    float *d_fb1 = nullptr, *d_fb2 = nullptr, *d_fb3 = nullptr;
    int hidden = 0;
    double flops = 0.0;                          // algorithmic FLOPs of the three conv blocks per window
};

// One captured form of the update: [incremental?][with profiling stamps?].
struct GraphVar {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t append_node = nullptr;       // the kernels that read the caller's new-sample buffer
    cudaGraphNode_t ring16_node = nullptr;
    cudaGraphNode_t agg_node = nullptr;          // writes the caller's final-samples buffer
    cudaGraphNode_t scores_node = nullptr;       // memcpy of the scores into the caller's buffer
    bool append_fused = false;                   // append_node is k_snapshot_append (a1 + a2 in one kernel)
    int nodes = 0;
    const float* cap_in = nullptr;
    float* cap_scores = nullptr;
    float* cap_final = nullptr;
    AggParams agg;                               // the aggregation node's argument as captured
    Prof prof;                                   // stamped variants: kernel labels in launch order
};

struct gw_pipeline {
    HandleBase base;
    gw_stream* s = nullptr;
    gw_deepclean* dc = nullptr;
    gw_bbh* bbh = nullptr;
    GraphVar var[2][2];                          // [incremental zones][profiling stamps]
    unsigned long long* d_stamps = nullptr;      // [kMaxStamps][2]
    const Prof* last_prof = nullptr;
    float *d_in = nullptr, *d_scores = nullptr, *d_final = nullptr;   // staging for gw_step_host
    float* d_in2[2] = {nullptr, nullptr};        // gw_step_host_async: double-buffered input staging,
    cudaStream_t copy_stream = nullptr;          // filled on an internal copy stream while the previous step computes
    cudaEvent_t in_done[2] = {nullptr, nullptr}, in_free[2] = {nullptr, nullptr};
    int64_t async_calls = 0;
};

// Incremental path (D13): how many OUTPUT positions of each layer differ from the previous update's value at
// the same absolute position.  `left[i]`: positions [0, left) whose receptive field reaches the left window edge (where
// this window pads with zeros and the previous one held data); `right[i]`: the last positions, which see the S new
// samples or the right window edge.  Recurrences for stride 2, odd k = 2p + 1, padding p (output_padding 1):
//   Conv1d            y[l] reads x[2l - p .. 2l + p]:            e' = floor((e - 1 + p)/2) + 1,  r' = floor((r + p)/2),  new' = new/2
//   ConvTranspose1d   y[m] reads x[ceil((m-p)/2) .. floor((m+p)/2)]:  e' = 2e - 1 + p,           r' = 2r + p,           new' = 2 new
// with e = r = 0, new = S at the network input.  right[i] = new_i + r_i.
static int incremental_zones(const std::vector<HostLayer>& layers, int n_layers, int S, std::vector<int>& left,
                             std::vector<int>& right) {
    int e = 0, r = 0, nw = S;
    left.assign(n_layers, 0); right.assign(n_layers, 0);
    for (int i = 0; i < n_layers; ++i) {
        const HostLayer& H = layers[i];
        if (H.stride != 2 || (H.k & 1) == 0) return fail(GW_EINVAL, "incremental path needs stride-2 layers with odd k");
        const int p = H.k / 2;
        if (H.kind == GW_CONV) {
            if (nw % 2) return fail(GW_EINVAL, "incremental path needs the stride to be a multiple of 2^(encoder depth)");
            e = (e - 1 + p) / 2 + 1; r = (r + p) / 2; nw /= 2;
        } else {
            e = 2 * e - 1 + p; r = 2 * r + p; nw *= 2;
        }
        left[i] = e; right[i] = nw + r;
    }
    return GW_OK;
}

extern "C" int gw_incremental_zones(const gw_conv_layer* layers, int n_layers, int stride, int* left, int* right) {
    if (!layers || !left || !right || n_layers < 1 || stride < 1) return fail(GW_EINVAL, "gw_incremental_zones: bad argument");
    std::vector<HostLayer> H(n_layers);
    for (int i = 0; i < n_layers; ++i) {
        H[i].kind = layers[i].kind; H[i].k = layers[i].k; H[i].stride = layers[i].stride;
        H[i].cin = layers[i].cin; H[i].cout = layers[i].cout;
    }
    std::vector<int> l, r;
    if (int rc = incremental_zones(H, n_layers, stride, l, r)) return rc;
    for (int i = 0; i < n_layers; ++i) { left[i] = l[i]; right[i] = r[i]; }
    return GW_OK;
}

// ------------------------------------------------------------------------------ GEMM layer build
// Builds B (weights in segment order), bias, the segment table and the tensor maps for one layer.
// tap(a, par, r): index j of the filter tap that connects A-view row shift a, column half `par`
// (position parity inside a pair row; always 0 for GK_DEC) to output column half r; <0 or >=k: none.
// ring_count != null: the input is a mirror ring (every row stored twice, 2 a_rows rows per batch item) whose window
// starts at row (*ring_count mod ring_W) / (ring_W / a_rows); out_ring: so is the output (incremental path).
static int build_gemm_layer(GemmLayer& gl, GemmKind gk, const HostLayer* dets, int n_det, int fmt, const gw_options& opt,
                            const void* in, int in_L, int cin_p, void* out, int cout_p, int batch, int epi,
                            int head_hidden = 0, const long long* ring_count = nullptr, int ring_W = 0,
                            bool out_ring = false, long long seg_T = 0, int seg_S = 0, int ring_S = 0) {
    const HostLayer& H0 = dets[0];
    ConvGemmParams& p = gl.g.p;
    memset(&p, 0, sizeof p);
    const int halves_in = gk == GK_DEC ? 1 : 2;       // A view packs position pairs?
    const int halves_out = gk == GK_ENC ? 1 : 2;      // N packs (even | odd) outputs?
    p.a_cols = halves_in * cin_p;
    p.a_rows = in_L / halves_in;
    p.a_rows_tm = ring_count ? 2 * p.a_rows : p.a_rows;     // mirror ring: every sample stored twice
    p.a_count = ring_count;
    p.a_ring_W = ring_W;
    p.a_ring_div = ring_count ? ring_W / p.a_rows : 1;
    p.M = p.a_rows;
    p.N = halves_out * cout_p;
    p.n_det = n_det;
    p.fmt = fmt;
    p.epi = epi;
    p.act = H0.act;
    if (ring_count && (ring_W % p.a_rows)) return fail(GW_EINVAL, "ring input: window %d is not a multiple of the layer's %d rows", ring_W, p.a_rows);
    if (out_ring && (!ring_count || epi != EPI_STORE || p.M % kTileM))
        return fail(GW_EINVAL, "incremental path: layer with %d rows cannot write a ring (needs a ring input and rows %% 128 == 0)", p.M);
    p.out_ring_div = out_ring ? ring_W / p.M : 0;
    if (p.N > 256 || p.N % 32) return fail(GW_EINVAL, "GEMM N = %d unsupported (must be a multiple of 32, <= 256)", p.N);
    if (epi == EPI_FINAL && p.N != 64) return fail(GW_EINVAL, "fused final layer needs GEMM N = 64, got %d", p.N);
    if (epi == EPI_STORE && p.N != 32 && p.N != 64 && p.N != 128 && p.N != 256)
        return fail(GW_EINVAL, "GEMM N = %d unsupported by the store epilogue (32, 64, 128 or 256)", p.N);
    if (p.a_cols % kSegK) return fail(GW_EINVAL, "A view width %d not a multiple of 64", p.a_cols);
    auto tap = [&](int a, int par, int r) -> int {
        switch (gk) {
            case GK_ENC: return 2 * a + par + H0.pad_l;               // x index 2l + j - pad = 2(l+a) + par
            case GK_DEC: return ((r + H0.pad_l - 2 * a));             // m = 2l + j - pad, m = 2q + r, l = q + a
            default:     return 2 * a + par - r + H0.pad_l;           // x index (2m + r) + j - pad = 2(m+a) + par
        }
    };
    // segment table, ordered column block outer / row shift inner (the order the kernel issues MMAs in)
    int n_seg = 0, a_lo = 99, a_hi = -99;
    std::vector<int> seg_a, seg_cb;
    p.n_cb = p.a_cols / kSegK;
    if (p.n_cb > kMaxCb) return fail(GW_EINVAL, "A view width %d too wide", p.a_cols);
    for (int cb = 0; cb < p.n_cb; ++cb)
        for (int a = -8; a <= 8; ++a) {
            bool any = false;
            for (int kk = 0; kk < kSegK && !any; ++kk) {
                const int col = cb * kSegK + kk, par = col / cin_p, ci = col % cin_p;
                if (ci >= H0.cin) continue;
                for (int r = 0; r < halves_out; ++r) {
                    const int j = tap(a, par, r);
                    if (j >= 0 && j < H0.k) any = true;
                }
            }
            if (any) {
                seg_a.push_back(a); seg_cb.push_back(cb); ++n_seg;
                if (a < a_lo) a_lo = a;
                if (a > a_hi) a_hi = a;
            }
        }
    if (n_seg > kMaxSeg || n_seg < 1) return fail(GW_EINVAL, "layer needs %d K segments (max %d)", n_seg, kMaxSeg);
    p.n_seg = n_seg;
    p.a_min = a_lo;
    p.n_shift = a_hi - a_lo + 1;
    if (p.n_shift > kMaxShift) return fail(GW_EINVAL, "layer needs %d row shifts (max %d)", p.n_shift, kMaxShift);
    p.slab_rows = kTileM + p.n_shift - 1;
    p.tile_stride = epi == EPI_FINAL ? kTileM - 2 : kTileM;     // EPI_FINAL: one halo row on each side
    p.tile_row0 = epi == EPI_FINAL ? -1 : 0;
    p.tiles_m = (p.M + p.tile_stride - 1) / p.tile_stride;
    p.v_tiles = p.v_left = p.tiles_m;                           // whole windows
    memset(p.seg_of, 0xff, sizeof p.seg_of);
    for (int s = 0; s < n_seg; ++s) {
        p.seg_shift[s] = static_cast<int8_t>(seg_a[s]);
        p.seg_col[s] = static_cast<int16_t>(seg_cb[s] * kSegK);
        p.seg_of[seg_cb[s]][seg_a[s] - a_lo] = static_cast<int8_t>(s);
    }
    // structural zeros of each segment (which K steps / which half of N any filter tap reaches at all)
    if (opt.skip_zeros && epi != EPI_POOL && epi != EPI_POOL_HEAD) {
        for (int s = 0; s < n_seg; ++s) {
            bool k01 = false, lower = false, upper = false;
            for (int kk = 0; kk < kSegK; ++kk) {
                const int col = seg_cb[s] * kSegK + kk, par = col / cin_p, ci = col % cin_p;
                if (ci >= H0.cin) continue;
                for (int r = 0; r < halves_out; ++r) {
                    const int j = tap(seg_a[s], par, r);
                    if (j < 0 || j >= H0.k) continue;
                    if (kk < 32) k01 = true;
                    (r == 0 ? lower : upper) = true;
                }
            }
            const unsigned long long bit = 1ull << (seg_cb[s] * kMaxShift + (seg_a[s] - a_lo));
            if (halves_out == 2 && upper && !lower && s > 0 && (p.N / 2) % 16 == 0) p.mask_nu |= bit;   // never the tile's first MMA
            else if (!k01) p.mask_k2 |= bit;
        }
    }
    // weights and bias
    const size_t ktot = static_cast<size_t>(n_seg) * kSegK;
    std::vector<uint16_t> B(static_cast<size_t>(n_det) * p.N * ktot, 0);
    std::vector<float> bias(static_cast<size_t>(n_det) * p.N, 0.f);
    for (int d = 0; d < n_det; ++d) {
        const HostLayer& H = dets[d];
        for (int r = 0; r < halves_out; ++r)
            for (int co = 0; co < H.cout; ++co) {
                const int n = r * cout_p + co;
                bias[static_cast<size_t>(d) * p.N + n] = static_cast<float>(H.b[co]);
                for (int s = 0; s < n_seg; ++s)
                    for (int kk = 0; kk < kSegK; ++kk) {
                        const int col = seg_cb[s] * kSegK + kk, par = col / cin_p, ci = col % cin_p;
                        if (ci >= H.cin) continue;
                        const int j = tap(seg_a[s], par, r);
                        if (j < 0 || j >= H.k) continue;
                        B[(static_cast<size_t>(d) * p.N + n) * ktot + static_cast<size_t>(s) * kSegK + kk] =
                            to_storage_bits(H.W(co, ci, j), fmt);
                    }
            }
    }
    CU_TRY(cudaMalloc(&gl.d_B, B.size() * 2));
    CU_TRY(cudaMemcpy(gl.d_B, B.data(), B.size() * 2, cudaMemcpyHostToDevice));
    CU_TRY(cudaMalloc(&gl.d_bias, bias.size() * 4));
    CU_TRY(cudaMemcpy(gl.d_bias, bias.data(), bias.size() * 4, cudaMemcpyHostToDevice));
    p.A = in; p.B = gl.d_B; p.bias = gl.d_bias; p.out = out;
    if (seg_T > 0) {
        // offline first layer: `in` = [n_det][seg_T][cin_p]; window j starts seg_S positions after window j - 1
        p.a_4d = 1;
        if (int rc = make_tmap4(&p.tmA, in, fmt, p.a_cols, p.a_rows, n_det, batch / n_det, p.a_cols,
                                static_cast<uint64_t>(seg_T) * cin_p, static_cast<uint64_t>(seg_S) * cin_p, p.slab_rows)) return rc;
    } else if (int rc = make_tmap(&p.tmA, in, fmt, p.a_cols, p.a_rows_tm, batch, p.a_cols, static_cast<uint64_t>(p.a_rows_tm) * p.a_cols, p.slab_rows)) return rc;
    if (epi == EPI_STORE) {  // output [batch][M][N] ([batch][2M][N] as a mirror ring): one 32-row x min(N, 64)-column box per epilogue-warp store
        const uint64_t out_rows = out_ring ? 2 * static_cast<uint64_t>(p.M) : p.M;
        if (int rc = make_tmap(&p.tmOut, out, fmt, p.N, out_rows, batch, p.N, out_rows * p.N, 32, p.N >= 64 ? 64 : 32)) return rc;
    }
    if (ring_count && ring_S > 0 && ring_W % ring_S == 0 && ring_S % p.a_ring_div == 0 && seg_T == 0) {
        // ring input: a tensor map per window head (see ConvGemmParams::tmA_heads), so that rows outside the window are
        // TMA's zero fill.  The CTA-pair kernel needs them; the one-CTA kernel would otherwise clear those rows in shared
        // memory from its MMA warp, with a proxy fence per column block in front of the MMAs -- every tile of a zone launch
        // lies on a window edge and paid it (GW_TRACE at n = 512: 12.7 k cycles per tile in the MMA warp against 2.4 k)
        const int n_heads = ring_W / ring_S;
        std::vector<CUtensorMap> heads(n_heads);
        for (int h = 0; h < n_heads; ++h) {
            const size_t off_rows = static_cast<size_t>(h) * ring_S / p.a_ring_div;
            const uint16_t* base = static_cast<const uint16_t*>(in) + off_rows * p.a_cols;
            if (int rc = make_tmap(&heads[h], base, fmt, p.a_cols, p.a_rows, batch, p.a_cols,
                                   static_cast<uint64_t>(p.a_rows_tm) * p.a_cols, p.slab_rows)) return rc;
        }
        CU_TRY(cudaMalloc(&gl.d_heads, sizeof(CUtensorMap) * n_heads));
        CU_TRY(cudaMemcpy(gl.d_heads, heads.data(), sizeof(CUtensorMap) * n_heads, cudaMemcpyHostToDevice));
        p.tmA_heads = gl.d_heads;
        p.head_div = ring_S;
    }
    gl.g.batch = batch;
    gl.g.pdl = opt.pdl;
    p.head_hidden = head_hidden;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    p.two_sm = opt.two_sm;                             // a request: the plan keeps it only where the pair kernel applies
    if (!conv_gemm_plan(gl.g, sms)) return fail(GW_EINVAL, "conv GEMM layer does not fit in shared memory");
    if (int rc = make_tmap(&p.tmB, gl.d_B, fmt, ktot, p.N, n_det, ktot, static_cast<uint64_t>(p.N) * ktot, p.two_sm ? 128 : p.N)) return rc;
    if (p.mask_nu)
        if (int rc = make_tmap(&p.tmBh, gl.d_B, fmt, ktot, p.N, n_det, ktot, static_cast<uint64_t>(p.N) * ktot, p.N / 2)) return rc;
    gl.impl = opt.conv_impl;
#ifdef GW_TRACE
    CU_TRY(cudaMalloc(&p.trace, 148 * 16 * 8));
    CU_TRY(cudaMemset(p.trace, 0, 148 * 16 * 8));
#endif
    return GW_OK;
}

// Incremental variant of a built layer: the same operands, work list = the tiles that cover the first `left_rows`
// and the last `right_rows` GEMM rows of every batch item (all tiles when the two zones meet).
static int make_incremental_variant(GemmLayer& gl, int left_rows, int right_rows) {
    gl.gi = gl.g;
    ConvGemmParams& p = gl.gi.p;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // CTA-pair layers (ring input through per-head tensor maps): both zones in ONE tile per batch item when they fit, the
    // pair working on two batch items -- half the tiles (and half the streamed weights) of a tile per zone
    if (p.two_sm && p.tmA_heads && (gl.g.batch / p.n_det) % 2 == 0) {
        const int nl = round_up(left_rows + p.n_shift - 1, 8), nr = round_up(right_rows + p.n_shift - 1, 8);
        if (nl + nr <= kTileM && left_rows + right_rows < p.M) {
            // as many batch items per tile as fit (and as divide the batch): 2 at S = 512, 4 at S = 256
            int k = kTileM / (nl + nr);
            while (k > 1 && (gl.g.batch / p.n_det) % (2 * k)) --k;
            const int n_heads = p.a_ring_W / p.head_div;
            std::vector<CUtensorMap> heads(n_heads), heads_r(n_heads);
            for (int h = 0; h < n_heads; ++h) {
                const size_t off_rows = static_cast<size_t>(h) * p.head_div / p.a_ring_div;
                const uint16_t* base = static_cast<const uint16_t*>(p.A) + off_rows * p.a_cols;
                if (int rc = make_tmap(&heads[h], base, p.fmt, p.a_cols, p.a_rows, gl.g.batch, p.a_cols,
                                       static_cast<uint64_t>(p.a_rows_tm) * p.a_cols, nl)) return rc;
                if (int rc = make_tmap(&heads_r[h], base, p.fmt, p.a_cols, p.a_rows, gl.g.batch, p.a_cols,
                                       static_cast<uint64_t>(p.a_rows_tm) * p.a_cols, nr)) return rc;
            }
            CU_TRY(cudaMalloc(&gl.d_heads_left, sizeof(CUtensorMap) * n_heads));
            CU_TRY(cudaMemcpy(gl.d_heads_left, heads.data(), sizeof(CUtensorMap) * n_heads, cudaMemcpyHostToDevice));
            CU_TRY(cudaMalloc(&gl.d_heads_right, sizeof(CUtensorMap) * n_heads));
            CU_TRY(cudaMemcpy(gl.d_heads_right, heads_r.data(), sizeof(CUtensorMap) * n_heads, cudaMemcpyHostToDevice));
            p.tmA_heads_left = gl.d_heads_left;
            p.tmA_heads_right = gl.d_heads_right;
            p.pk_nl = nl; p.pk_nr = nr; p.pk_k = k; p.pk_left = left_rows; p.pk_right = right_rows;
            p.v_left = 0; p.v_tiles = 1;                // one (packed) tile per pk_k batch items
            if (conv_gemm_plan(gl.gi, sms) && gl.gi.p.two_sm) { gl.has_inc = true; return GW_OK; }
            gl.gi = gl.g;                               // does not fit: the unpacked work list below
        }
    }
    const int ts = p.tile_stride;                       // tile t produces rows [t ts, t ts + ts)
    int v_left = (left_rows + ts - 1) / ts;
    int first_right = (p.M - right_rows) / ts;
    if (first_right < 0) first_right = 0;
    if (v_left > p.tiles_m) v_left = p.tiles_m;
    if (first_right <= v_left) { p.v_left = p.v_tiles = p.tiles_m; }
    else { p.v_left = v_left; p.v_tiles = v_left + (p.tiles_m - first_right); }
    // same operand layout (resident / streamed weights, CTA pair or not: the weight tensor map depends on it); only the
    // tiles-per-stage choice may differ.  A pair layer whose zones give an odd tile count gets one more left tile.
    if (p.two_sm && (p.v_tiles & 1)) { p.v_left += 1; p.v_tiles += 1; }
    if ((p.epi == EPI_STORE || p.epi == EPI_FINAL) && p.v_tiles < p.tiles_m) { p.z_left = left_rows; p.z_right = right_rows; }
    conv_gemm_plan(gl.gi, sms);
    gl.has_inc = true;
    return GW_OK;
}

#ifdef GW_TRACE
// Diagnostic builds: mean over CTAs of the per-role wait counters of the last launch of a layer.
static void trace_report(const GemmLayer& gl) {
    const ConvGemmParams& p = gl.g.p;
    if (!p.trace) return;
    std::vector<long long> h(148 * 16);
    cudaMemcpy(h.data(), p.trace, h.size() * 8, cudaMemcpyDeviceToHost);
    double m[16] = {0};
    int n = 0;
    for (int b = 0; b < 148; ++b) {
        if (h[b * 16 + 7] == 0) continue;
        ++n;
        for (int i = 0; i < 16; ++i) m[i] += static_cast<double>(h[b * 16 + i]);
    }
    if (!n) return;
    for (double& v : m) v /= n;
    fprintf(stderr, "[trace] %-10s N=%3d | producer: a_empty %7.0f b_empty %7.0f total %7.0f | mma: tmem_empty %7.0f a_full %7.0f "
                    "b_full %7.0f stg_full %7.0f total %7.0f | epi(w2): tmem_full %7.0f store_rd %7.0f fin_full %7.0f total %7.0f\n",
            gl.name.c_str(), p.N, m[0], m[1], m[2], m[3], m[4], m[5], m[6], m[7], m[8], m[9], m[10], m[11]);
}
#endif

// Shared-memory traffic of one launch of a conv GEMM layer, summed over all SMs, by the accounting of DESIGN.md
// section 7: per 128-row tile the tensor core reads 4 KiB of A plus 32 N bytes of B per MMA (half of B per SM in the
// CTA-pair kernel), TMA writes the A slabs (and, when weights are streamed, the weight blocks) and the epilogue
// writes its staged output once and TMA reads it once.  Divided by 128 B/clk/SM x SMs x clock it gives the
// shared-memory roofline the thin layers sit on.
static double gemm_smem_bytes(const GemmLaunch& g, int batch) {
    const ConvGemmParams& p = g.p;
    const int n_items = batch / p.n_det;
    int n_half = 0, n_k2 = 0;
    for (unsigned long long m = p.mask_nu; m; m &= m - 1) ++n_half;
    for (unsigned long long m = p.mask_k2; m; m &= m - 1) ++n_k2;
    const double b_per_mma = 32.0 * p.N * (p.two_sm ? 0.5 : 1.0);
    double mma = 4.0 * (p.n_seg - n_half - n_k2) * (4096.0 + b_per_mma)             // full segments: four K steps
               + 4.0 * n_half * (4096.0 + b_per_mma / 2) + 2.0 * n_k2 * (4096.0 + b_per_mma);
    double fill = static_cast<double>(p.n_cb) * p.slab_rows * 128.0;
    if (!p.b_resident) fill += static_cast<double>(p.n_seg) * p.N * 128.0 * (p.two_sm ? 0.5 : 1.0);
    double epi = 0.0;
    if (p.epi == EPI_STORE) epi = 2.0 * 128.0 * p.N * 2.0;                            // staged once, read once by the TMA store
    if (p.epi == EPI_FINAL) { epi = 128.0 * 128.0; mma += 10.0 * (4096.0 + 32.0 * 16); }   // activated tile + second chain
    return (mma + fill + epi) * static_cast<double>(p.v_tiles) * n_items * p.n_det / (p.pk_k > 1 ? p.pk_k : 1);
}

static void run_gemm(const GemmLayer& gl, LaunchCtx& cx, bool inc = false, int batch_override = 0) {
    GemmLaunch g = (inc && gl.has_inc) ? gl.gi : gl.g;
    if (batch_override) g.batch = batch_override;
    // algorithmic FLOPs this launch executes: the rows of its tiles (all of them, or the recomputed zones)
    const double rows = static_cast<double>(g.p.v_tiles) * g.p.tile_stride;
    double frac = rows >= g.p.M ? 1.0 : rows / g.p.M;
    if (g.p.pk_k > 1) frac /= g.p.pk_k;                 // packed zones: one tile per pk_k batch items
    g.p.stamp = cx.next(gl.name, gl.flops * g.batch * frac, gemm_smem_bytes(g, g.batch));
    cx.check(gl.impl == GW_IMPL_UMMA ? launch_conv_gemm_umma(g, cx.st) : launch_conv_gemm_simt(g, cx.st));
}

static void free_gemm(GemmLayer& gl) {
    cudaFree(gl.d_B); cudaFree(gl.d_bias); cudaFree(gl.d_heads); cudaFree(gl.d_heads_left); cudaFree(gl.d_heads_right);
    gl.d_B = nullptr; gl.d_bias = nullptr; gl.d_heads = nullptr; gl.d_heads_left = nullptr; gl.d_heads_right = nullptr;
}

// =============================================================================== snapshotter
extern "C" int gw_stream_create(gw_stream** out, int n_streams, int channels, int fs, int window, int stride) {
    if (!out) return fail(GW_EINVAL, "out is NULL");
    *out = nullptr;
    if (n_streams < 1 || channels < 1 || fs < 1 || window < 1 || stride < 1 || stride > window)
        return fail(GW_EINVAL, "gw_stream_create: need n_streams, channels, fs >= 1 and 1 <= stride <= window");
    if (int rc = check_device()) return rc;
    gw_stream* s = new gw_stream();
    s->n = n_streams; s->C = channels; s->fs = fs; s->W = window; s->S = stride;
    const size_t bytes = static_cast<size_t>(n_streams) * channels * window * sizeof(float);
    cudaError_t e = cudaMalloc(&s->ring, bytes);
    if (e == cudaSuccess) e = cudaMemset(s->ring, 0, bytes);
    if (e == cudaSuccess) e = cudaMalloc(&s->d_count, sizeof(long long));
    if (e == cudaSuccess) e = cudaMemset(s->d_count, 0, sizeof(long long));
    if (e == cudaSuccess) e = cudaMalloc(&s->d_ticket, sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(s->d_ticket, 0, sizeof(unsigned));
    if (e != cudaSuccess) {
        cudaFree(s->ring); cudaFree(s->d_count); cudaFree(s->d_ticket);
        delete s;
        return fail(e == cudaErrorMemoryAllocation ? GW_ENOMEM : GW_ECUDA, "gw_stream_create: %s", cudaGetErrorString(e));
    }
    *out = s;
    return GW_OK;
}

extern "C" int gw_stream_destroy(gw_stream* s) {
    if (!s) return GW_OK;
    cudaFree(s->ring); cudaFree(s->d_count); cudaFree(s->d_ticket);
    s->base.magic = 0;
    delete s;
    return GW_OK;
}

static void ring16_append_enqueue(gw_deepclean* dc, const float* src, LaunchCtx& cx);

static int stream_update_checked(gw_stream* s) {
    if (s->dc && s->dc->cleaned_for != s->updates)
        return fail(GW_ESTATE, "gw_stream_update: update %lld has not been through gw_deepclean_forward + gw_cleaned_strain",
                    (long long)s->updates);
    return GW_OK;
}
static void stream_update_enqueue(gw_stream* s, const float* src, LaunchCtx& cx) {
    gw_deepclean* dc = s->dc;
    if (dc && dc->mirror && s->S % 4 == 0 && s->W % 4 == 0) {       // a1 + a2 in one launch
        cx.check(launch_snapshot_append(s->ring, src, dc->ring16, s->d_count, s->d_ticket, dc->d_rows_map, dc->d_pre, s->n,
                                        s->C, dc->n_det, dc->n_wit, s->W, s->S, dc->act_cols[0], dc->fmt,
                                        cx.next("snapshot_append"), cx.st));
        return;
    }
    cx.check(launch_append(s->ring, src, s->d_count, s->d_ticket, s->n * s->C, s->W, s->S, cx.next("append"), cx.st));
    if (dc) ring16_append_enqueue(dc, src, cx);
}

extern "C" int gw_stream_update(gw_stream* s, const float* new_samples_dev, void* stream) {
    if (!s || !new_samples_dev) return fail(GW_EINVAL, "gw_stream_update: NULL argument");
    CallScope scope(s);
    if (int rc = stream_update_checked(s)) return rc;
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    stream_update_enqueue(s, new_samples_dev, cx);
    CX_TRY(cx, "gw_stream_update");
    s->updates += 1;
    return GW_OK;
}

extern "C" int gw_stream_snapshot(gw_stream* s, float* out_dev, int64_t* first_index_host, void* stream) {
    if (!s || !out_dev) return fail(GW_EINVAL, "gw_stream_snapshot: NULL argument");
    CallScope scope(s);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    CU_TRY(launch_snapshot(s->ring, out_dev, s->d_count, s->n * s->C, s->W, st));
    CU_TRY(cudaStreamSynchronize(st));
    if (first_index_host) *first_index_host = s->updates * static_cast<int64_t>(s->S) - s->W;
    return GW_OK;
}

extern "C" int64_t gw_stream_count(const gw_stream* s) { return s ? s->updates * static_cast<int64_t>(s->S) : 0; }

// ================================================================================= DeepClean
static int validate_dc_layer(const HostLayer& H, bool last) {
    if (H.stride != 2 || (H.k & 1) == 0) return fail(GW_EINVAL, "DeepClean layers need stride 2 and odd k");
    if (H.kind == GW_CONV && (H.pad_l != H.k / 2 || H.pad_r != H.k / 2)) return fail(GW_EINVAL, "Conv1d needs pad = k/2");
    if (H.kind == GW_CONVT && (H.pad_l != H.k / 2 || H.pad_r != 1)) return fail(GW_EINVAL, "ConvTranspose1d needs padding k/2, output_padding 1");
    if (H.pool != 1) return fail(GW_EINVAL, "DeepClean layers have no pooling");
    if (last && (H.kind != GW_CONVT || H.cout != 1 || H.act != GW_ACT_NONE || H.k > 7))
        return fail(GW_EINVAL, "last DeepClean layer must be a linear ConvTranspose1d with one output channel, k <= 7");
    return GW_OK;
}

extern "C" int gw_deepclean_destroy(gw_deepclean* dc) {
    if (!dc) return GW_OK;
    for (auto& g : dc->gemm) free_gemm(g);
    for (void* a : dc->act) cudaFree(a);
    cudaFree(dc->ring16); cudaFree(dc->seg16);
    cudaFree(dc->d_wt_final); cudaFree(dc->d_b_final); cudaFree(dc->d_fin_B); cudaFree(dc->pred); cudaFree(dc->acc); cudaFree(dc->nhat);
    cudaFree(dc->d_hann); cudaFree(dc->d_inv_wsum); cudaFree(dc->d_rows_map); cudaFree(dc->d_strain_rows);
    cudaFree(dc->d_pre); cudaFree(dc->d_post);
    cudaFree(dc->final_buf); cudaFree(dc->d_fir); cudaFree(dc->d_hist);
    if (dc->s && dc->s->dc == dc) dc->s->dc = nullptr;
    dc->base.magic = 0;
    delete dc;
    return GW_OK;
}

static int deepclean_build(gw_deepclean* dc, gw_stream* s, const gw_dc_spec* spec) {
    const int W = s->W, S = s->S;
    const int nl = spec->n_layers, nd = spec->n_det;
    const gw_options& opt = dc->opt;
    dc->host.resize(static_cast<size_t>(nd) * nl);
    for (int d = 0; d < nd; ++d)
        for (int i = 0; i < nl; ++i) {
            if (int rc = fold_layer(spec->layers[d * nl + i], dc->host[d * nl + i])) return rc;
            const HostLayer &H = dc->host[d * nl + i], &H0 = dc->host[i];
            if (int rc = validate_dc_layer(H, i == nl - 1)) return rc;
            if (H.kind != H0.kind || H.cin != H0.cin || H.cout != H0.cout || H.k != H0.k || H.act != H0.act)
                return fail(GW_EINVAL, "detectors must share the layer shapes");
        }
    if (dc->host[0].cin != spec->n_witness) return fail(GW_EINVAL, "first layer cin != n_witness");
    // padded channel counts: consumer decides (pair views need multiples of 32, ConvT inputs multiples of 64)
    std::vector<int> cpad(nl + 1);
    for (int i = 0; i <= nl; ++i) {
        const int c = i == 0 ? dc->host[0].cin : dc->host[i - 1].cout;
        if (i == nl) { cpad[i] = 1; break; }
        const bool gemm_consumer = i < nl - 1;
        cpad[i] = round_up(c, (gemm_consumer && dc->host[i].kind == GW_CONVT) ? 64 : 32);
    }
    // lengths
    std::vector<int> len(nl + 1);
    len[0] = W;
    for (int i = 0; i < nl; ++i) {
        const HostLayer& H = dc->host[i];
        if (H.kind == GW_CONV) {
            if (len[i] % 2) return fail(GW_EINVAL, "window length must be divisible by 2^(number of encoder layers)");
            len[i + 1] = len[i] / 2;
        } else {
            len[i + 1] = len[i] * 2;
        }
        if (i > 0 && dc->host[i].cin != dc->host[i - 1].cout) return fail(GW_EINVAL, "layer %d cin mismatch", i);
    }
    if (len[nl] != W) return fail(GW_EINVAL, "network output length %d != window %d", len[nl], W);
    const int batch = s->n * nd;
    dc->batch = batch;
    dc->act.assign(nl, nullptr);
    dc->act_rows.assign(nl, 0); dc->act_cols.assign(nl, 0);
    // The 16-bit mirror ring replaces the per-update gather when window positions pair up with ring slots
    // (even stride => even head) and the first layer is a Conv1d; otherwise the window is re-gathered.
    dc->mirror = !dc->offline && (S % 2 == 0) && (W % 2 == 0) && dc->host[0].kind == GW_CONV;
    // offline: the first layer reads overlapping windows of the converted segment through a 4-D tensor map when
    // window starts fall on position pairs (even stride); otherwise every window is gathered (k_gather)
    const bool direct_seg = dc->offline && (S % 2 == 0) && (W % 2 == 0) && dc->host[0].kind == GW_CONV &&
                            opt.conv_impl == GW_IMPL_UMMA;
    // The last GEMM layer (ConvTranspose1d -> <= 32 channels, tanh) and the final 1-channel ConvTranspose1d
    // (k = 7) run as ONE kernel when they have the standard shape: the 16-bit activation between them is
    // never written (at C3 that round trip is 2 x 1 MiB per detector-window, more than the layer's input).
    {
        const HostLayer &Hp = dc->host[nl - 2], &Hf = dc->host[nl - 1];
        dc->fused_tail = opt.fuse_tail && opt.conv_impl == GW_IMPL_UMMA && nl >= 3 && Hp.kind == GW_CONVT &&
                         Hp.act == GW_ACT_TANH && cpad[nl - 1] == 32 && Hf.k == 7 && Hf.pad_l == 3;
    }
    // Incremental path (D13): every stored activation is a mirror ring over absolute position; an update recomputes
    // the left-edge and right-edge rows only.
    std::vector<int> z_left, z_right;
    dc->inc = false;
    if (opt.incremental) {
        if (dc->offline) return fail(GW_EINVAL, "incremental path: streaming handles only");
        if (!dc->mirror || !dc->fused_tail || opt.conv_impl != GW_IMPL_UMMA)
            return fail(GW_EINVAL, "incremental path needs an even stride and window, a Conv1d first layer, the fused tail and GW_IMPL_UMMA");
        std::vector<HostLayer> one(dc->host.begin(), dc->host.begin() + nl);
        if (int rc = incremental_zones(one, nl, S, z_left, z_right)) return rc;
        int min_len = W;
        for (int i = 0; i <= nl; ++i) if (len[i] < min_len) min_len = len[i];
        const int depth_div = W / min_len;                  // 2^(encoder depth)
        if (S % depth_div || W % (depth_div * kTileM))
            return fail(GW_EINVAL, "incremental path needs stride %% %d == 0 and window %% %d == 0 (got %d, %d)", depth_div,
                        depth_div * kTileM, S, W);
        dc->inc = true;
    }
    for (int i = 0; i < nl; ++i) {                  // act[i] = input of layer i
        dc->act_rows[i] = len[i]; dc->act_cols[i] = cpad[i];
        if (i == nl - 1 && dc->fused_tail) continue;  // never materialised
        size_t bytes = static_cast<size_t>(batch) * len[i] * cpad[i] * 2;
        void** dst = &dc->act[i];
        if (i == 0 && dc->mirror) { bytes *= 2; dst = &dc->ring16; }
        else if (dc->inc) bytes *= 2;                 // mirror ring: every row twice
        if (i == 0 && direct_seg) { bytes = static_cast<size_t>(nd) * dc->off_T * cpad[0] * 2; dst = &dc->seg16; }
        CU_TRY(cudaMalloc(dst, bytes));
        CU_TRY(cudaMemset(*dst, 0, bytes));
    }
    dc->gemm.resize(nl - 1);
    std::vector<HostLayer> per_det(nd);
    for (int i = 0; i < nl - 1; ++i) {
        for (int d = 0; d < nd; ++d) per_det[d] = dc->host[d * nl + i];
        const GemmKind gk = dc->host[i].kind == GW_CONV ? GK_ENC : GK_DEC;
        const bool from_ring = (i == 0 && dc->mirror) || dc->inc;
        const bool fin = i == nl - 2 && dc->fused_tail;
        const bool from_seg = i == 0 && direct_seg;
        const void* in = (i == 0 && dc->mirror) ? dc->ring16 : from_seg ? dc->seg16 : dc->act[i];
        if (int rc = build_gemm_layer(dc->gemm[i], gk, per_det.data(), nd, dc->fmt, opt, in,
                                      len[i], cpad[i], dc->act[i + 1], cpad[i + 1], batch, fin ? EPI_FINAL : EPI_STORE, 0,
                                      from_ring ? s->d_count : nullptr, from_ring ? W : 0, dc->inc && !fin,
                                      from_seg ? dc->off_T : 0, from_seg ? S : 0, S))
            return rc;
        dc->gemm[i].g.p.reverse = opt.snake ? (i & 1) : 0;
        dc->gemm[i].name = "gemm.dc" + std::to_string(i);
        // useful MACs: every (input position, tap, cin, cout) product of the layer definition
        const HostLayer& H = dc->host[i];
        const double lin = len[i];
        dc->gemm[i].flops = 2.0 * (H.kind == GW_CONV ? lin / 2 : lin) * H.k * H.cin * H.cout;
        if (fin) {                                   // the final layer's MACs run in this kernel too
            const HostLayer& Hf = dc->host[nl - 1];
            dc->gemm[i].flops += 2.0 * len[nl - 1] * Hf.k * Hf.cin * Hf.cout;
        }
    }
    // final layer on CUDA cores: wt[d][j][ci] fp32 holding storage-rounded weights
    {
        const HostLayer& H = dc->host[nl - 1];
        dc->final_K = H.k; dc->final_pad = H.pad_l; dc->final_cpad = cpad[nl - 1]; dc->final_L = len[nl - 1];
        std::vector<float> wt(static_cast<size_t>(nd) * H.k * cpad[nl - 1], 0.f), bf(nd);
        for (int d = 0; d < nd; ++d) {
            const HostLayer& Hd = dc->host[d * nl + nl - 1];
            for (int j = 0; j < H.k; ++j)
                for (int ci = 0; ci < H.cin; ++ci)
                    wt[(static_cast<size_t>(d) * H.k + j) * cpad[nl - 1] + ci] =
                        static_cast<float>(storage_to_double(to_storage_bits(Hd.W(0, ci, j), dc->fmt), dc->fmt));
            bf[d] = static_cast<float>(Hd.b[0]);
        }
        CU_TRY(cudaMalloc(&dc->d_wt_final, wt.size() * 4));
        CU_TRY(cudaMemcpy(dc->d_wt_final, wt.data(), wt.size() * 4, cudaMemcpyHostToDevice));
        CU_TRY(cudaMalloc(&dc->d_b_final, bf.size() * 4));
        CU_TRY(cudaMemcpy(dc->d_b_final, bf.data(), bf.size() * 4, cudaMemcpyHostToDevice));
    }
    const size_t wbytes = static_cast<size_t>(batch) * W * sizeof(float);
    CU_TRY(cudaMalloc(&dc->pred, wbytes));
    CU_TRY(cudaMemset(dc->pred, 0, wbytes));
    if (dc->fused_tail) {
        // The last layer as the B operand of a second MMA chain: N = 16 rows (r = 0..3 real: y[4m + r]),
        // K = 3 row shifts (a = -1, 0, 1) x 64 columns (par x 32 + ci: x[2(m + a) + par][ci]); the tap that
        // connects them is j = r + pad - 4a - 2 par (o = 2l + j - pad, D3).
        const HostLayer& H = dc->host[nl - 1];
        const int ktot = 3 * kSegK;
        std::vector<uint16_t> FB(static_cast<size_t>(nd) * 16 * ktot, 0);
        for (int d = 0; d < nd; ++d) {
            const HostLayer& Hd = dc->host[d * nl + nl - 1];
            for (int r = 0; r < 4; ++r)
                for (int a = -1; a <= 1; ++a)
                    for (int par = 0; par < 2; ++par) {
                        const int j = r + H.pad_l - 4 * a - 2 * par;
                        if (j < 0 || j >= H.k) continue;
                        for (int ci = 0; ci < H.cin; ++ci)
                            FB[(static_cast<size_t>(d) * 16 + r) * ktot + (a + 1) * kSegK + par * 32 + ci] =
                                to_storage_bits(Hd.W(0, ci, j), dc->fmt);
                    }
        }
        CU_TRY(cudaMalloc(&dc->d_fin_B, FB.size() * 2));
        CU_TRY(cudaMemcpy(dc->d_fin_B, FB.data(), FB.size() * 2, cudaMemcpyHostToDevice));
        ConvGemmParams& p = dc->gemm[nl - 2].g.p;
        if (int rc = make_tmap(&p.tmF, dc->d_fin_B, dc->fmt, ktot, 16, nd, ktot, static_cast<uint64_t>(16) * ktot, 16)) return rc;
        p.fin_b = dc->d_b_final; p.pred = dc->pred;
        p.pred_ring = dc->inc ? 1 : 0;
    }
    // gw_options.fuse_head: the first two encoder layers as one kernel (EPI_CHAIN, gw_conv_gemm.cu) -- whole-window
    // streaming handles whose layers 0 / 1 are the stride-2 Conv1d pair that kernel is written for (GEMM N 32 and 64, one
    // 64-column block, four row shifts from -2, resident weights, window edges as TMA zero fill)
    if (opt.fuse_head && !dc->inc && !dc->offline && opt.conv_impl == GW_IMPL_UMMA && nl >= 4 &&
        dc->host[0].kind == GW_CONV && dc->host[1].kind == GW_CONV) {
        const ConvGemmParams &p0 = dc->gemm[0].g.p, &p1 = dc->gemm[1].g.p;
        const bool edge_ok = p0.a_count == nullptr || p0.tmA_heads != nullptr;
        if (p0.epi == EPI_STORE && p1.epi == EPI_STORE && p0.act == ACT_TANH && p1.act == ACT_TANH && p0.N == 32 && p1.N == 64 &&
            p0.n_cb == 1 && p1.n_cb == 1 && p0.n_shift == 4 && p1.n_shift == 4 && p0.a_min == -2 && p1.a_min == -2 &&
            p0.b_resident && p1.b_resident && p1.n_seg == 4 && p1.mask_nu == 0 && p0.mask_nu == 0 && !p0.a_4d && edge_ok &&
            p1.a_rows * 2 == p0.M && p0.M % 2 == 0) {
            dc->chain = dc->gemm[0];                    // operands, segment table, input tensor maps of layer 0
            GemmLayer& c = dc->chain;
            c.has_inc = false;
            ConvGemmParams& p = c.g.p;
            p.epi = EPI_CHAIN;
            p.M2 = p1.M;
            const int n_super = (p.M2 + 124) / 125;
            p.tiles_m = p.v_tiles = p.v_left = 2 * n_super;
            p.tile_stride = kTileM; p.tile_row0 = 0;
            p.g_tiles = 0; p.out_bufs = 0;
            p.bias2 = dc->gemm[1].d_bias;
            p.out2 = dc->act[2];
            p.chain_k2 = static_cast<int>(p1.mask_k2 & ((1ull << kMaxShift) - 1));
            p.reverse = opt.snake ? 1 : 0;              // layer 2 walks forwards: end where it starts
            const size_t ktot2 = static_cast<size_t>(p1.n_seg) * kSegK;
            if (int rc = make_tmap(&p.tmF, dc->gemm[1].d_B, dc->fmt, ktot2, 64, nd, ktot2, 64 * ktot2, 64)) return rc;
            if (int rc = make_tmap(&p.tmOut, dc->act[2], dc->fmt, 64, p.M2, batch, 64, static_cast<uint64_t>(p.M2) * 64, 32, 32)) return rc;
            int dev = 0, sms = 148;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            p.two_sm = 0;
            if (conv_gemm_plan(c.g, sms) && c.g.p.b_resident) {
                c.name = "gemm.dc0+1";
                c.flops = dc->gemm[0].flops + dc->gemm[1].flops;
                c.d_B = nullptr; c.d_bias = nullptr; c.d_heads = nullptr; c.d_heads_left = nullptr; c.d_heads_right = nullptr;
                dc->has_chain = true;
            }
        }
    }
    if (dc->inc) {
        // zones in GEMM rows: an encoder row is one output position, a decoder row two (even | odd output), a row of the
        // fused tail four positions of the network output
        for (int i = 0; i < nl - 1; ++i) {
            const bool fin = i == nl - 2;
            const int per_row = fin ? 4 : (dc->host[i].kind == GW_CONV ? 1 : 2);
            const int zl = fin ? z_left[nl - 1] : z_left[i], zr = fin ? z_right[nl - 1] : z_right[i];
            if (int rc = make_incremental_variant(dc->gemm[i], (zl + per_row - 1) / per_row, (zr + per_row - 1) / per_row)) return rc;
        }
    }
    CU_TRY(cudaMalloc(&dc->acc, wbytes));
    CU_TRY(cudaMemset(dc->acc, 0, wbytes));
    CU_TRY(cudaMalloc(&dc->final_buf, static_cast<size_t>(batch) * S * sizeof(float)));
    // periodic Hann window and the reciprocal of the summed weights covering window position n:
    // wsum[n] = sum_{i >= 0, n + iS < W} w[n + iS]  (every sample with absolute index >= 0 has exactly
    // these windows over it, during warm-up as well: older windows would only add samples < 0).
    {
        std::vector<double> w(W);
        const double pi = 3.14159265358979323846;
        for (int n = 0; n < W; ++n) w[n] = 0.5 - 0.5 * cos(2.0 * pi * n / W);
        std::vector<float> wf(W), inv(W);
        for (int n = 0; n < W; ++n) {
            double sum = 0.0;
            for (int m = n; m < W; m += S) sum += w[m];
            wf[n] = static_cast<float>(w[n]);
            inv[n] = sum > 0.0 ? static_cast<float>(1.0 / sum) : 0.f;
        }
        CU_TRY(cudaMalloc(&dc->d_hann, W * 4));
        CU_TRY(cudaMemcpy(dc->d_hann, wf.data(), W * 4, cudaMemcpyHostToDevice));
        CU_TRY(cudaMalloc(&dc->d_inv_wsum, W * 4));
        CU_TRY(cudaMemcpy(dc->d_inv_wsum, inv.data(), W * 4, cudaMemcpyHostToDevice));
    }
    CU_TRY(cudaMalloc(&dc->d_rows_map, static_cast<size_t>(nd) * spec->n_witness * sizeof(int)));
    CU_TRY(cudaMemcpy(dc->d_rows_map, spec->witness_rows, static_cast<size_t>(nd) * spec->n_witness * sizeof(int), cudaMemcpyHostToDevice));
    CU_TRY(cudaMalloc(&dc->d_strain_rows, nd * sizeof(int)));
    CU_TRY(cudaMemcpy(dc->d_strain_rows, spec->strain_row, nd * sizeof(int), cudaMemcpyHostToDevice));
    {
        std::vector<float> pre(static_cast<size_t>(nd) * spec->n_witness * 2), post(static_cast<size_t>(nd) * 2);
        for (size_t i = 0; i < pre.size(); i += 2) { pre[i] = 0.f; pre[i + 1] = 1.f; }
        for (size_t i = 0; i < post.size(); i += 2) { post[i] = 1.f; post[i + 1] = 0.f; }
        CU_TRY(cudaMalloc(&dc->d_pre, pre.size() * 4));
        CU_TRY(cudaMemcpy(dc->d_pre, pre.data(), pre.size() * 4, cudaMemcpyHostToDevice));
        CU_TRY(cudaMalloc(&dc->d_post, post.size() * 4));
        CU_TRY(cudaMemcpy(dc->d_post, post.data(), post.size() * 4, cudaMemcpyHostToDevice));
    }
    CU_TRY(conv_gemm_prepare());
    return GW_OK;
}

// Pre/post-processing at the edges of DeepClean (PAPER.md:198 "preprocesses", :212 "postprocessed"; the paper
// never defines them: DESIGN.md reading A14): witness c of detector d enters the network as
// (x - wit_mean) / wit_std, and the aggregated estimate is subtracted as strain_std * nhat + strain_mean.
static int set_scaling(gw_deepclean* dc, const float* wit_mean, const float* wit_std, const float* strain_mean,
                       const float* strain_std) {
    const int nd = dc->n_det, nw = dc->n_wit;
    std::vector<float> pre(static_cast<size_t>(nd) * nw * 2), post(static_cast<size_t>(nd) * 2);
    for (int i = 0; i < nd * nw; ++i) {
        const double sd = wit_std ? wit_std[i] : 1.0;
        if (!(sd > 0.0) || !isfinite(sd)) return fail(GW_EINVAL, "witness std must be finite and > 0");
        pre[2 * i] = wit_mean ? wit_mean[i] : 0.f;
        pre[2 * i + 1] = wit_std ? static_cast<float>(1.0 / sd) : 1.f;
    }
    for (int d = 0; d < nd; ++d) {
        post[2 * d] = strain_std ? strain_std[d] : 1.f;
        post[2 * d + 1] = strain_mean ? strain_mean[d] : 0.f;
        if (!isfinite(post[2 * d]) || !isfinite(post[2 * d + 1])) return fail(GW_EINVAL, "strain scaling must be finite");
    }
    CU_TRY(cudaMemcpy(dc->d_pre, pre.data(), pre.size() * 4, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(dc->d_post, post.data(), post.size() * 4, cudaMemcpyHostToDevice));
    return GW_OK;
}

extern "C" int gw_deepclean_set_scaling(gw_deepclean* dc, const float* wit_mean, const float* wit_std,
                                        const float* strain_mean, const float* strain_std) {
    if (!dc) return fail(GW_EINVAL, "gw_deepclean_set_scaling: NULL handle");
    CallScope scope(dc);
    if (dc->s && dc->s->updates != 0)
        return fail(GW_ESTATE, "gw_deepclean_set_scaling: must be called before the first update (the state holds converted samples)");
    return set_scaling(dc, wit_mean, wit_std, strain_mean, strain_std);
}

// D11: causal FIR over the stream of emitted (final) estimate samples.
extern "C" int gw_deepclean_set_postfilter(gw_deepclean* dc, const float* taps_host, int n_taps) {
    if (!dc) return fail(GW_EINVAL, "gw_deepclean_set_postfilter: NULL handle");
    CallScope scope(dc);
    if (dc->offline) return fail(GW_EINVAL, "gw_deepclean_set_postfilter: streaming handles only");
    if (dc->s && dc->s->updates != 0)
        return fail(GW_ESTATE, "gw_deepclean_set_postfilter: must be called before the first update (the filter carries state)");
    if (!taps_host || n_taps == 0) {             // off
        cudaFree(dc->d_fir); cudaFree(dc->d_hist);
        dc->d_fir = nullptr; dc->d_hist = nullptr; dc->fir_n = 0;
        return GW_OK;
    }
    if (n_taps < 1 || n_taps > kMaxFir || n_taps - 1 > dc->s->S)
        return fail(GW_EINVAL, "post-filter needs 1 <= n_taps <= %d and n_taps - 1 <= stride", kMaxFir);
    for (int i = 0; i < n_taps; ++i)
        if (!isfinite(taps_host[i])) return fail(GW_EINVAL, "post-filter taps must be finite");
    cudaFree(dc->d_fir); cudaFree(dc->d_hist);
    dc->d_fir = nullptr; dc->d_hist = nullptr;
    const size_t hbytes = 2 * static_cast<size_t>(dc->batch) * (kMaxFir - 1) * sizeof(float);
    CU_TRY(cudaMalloc(&dc->d_fir, n_taps * sizeof(float)));
    CU_TRY(cudaMemcpy(dc->d_fir, taps_host, n_taps * sizeof(float), cudaMemcpyHostToDevice));
    CU_TRY(cudaMalloc(&dc->d_hist, hbytes));
    CU_TRY(cudaMemset(dc->d_hist, 0, hbytes));
    dc->fir_n = n_taps;
    return GW_OK;
}

extern "C" int gw_deepclean_create(gw_deepclean** out, gw_stream* s, const gw_dc_spec* spec, int dtype, const gw_options* opts) {
    if (!out) return fail(GW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!s || !spec || !spec->layers || !spec->witness_rows || !spec->strain_row) return fail(GW_EINVAL, "gw_deepclean_create: NULL argument");
    CallScope scope(s);
    if (dtype != GW_BF16 && dtype != GW_FP16) return fail(GW_EINVAL, "dtype must be GW_BF16 or GW_FP16");
    if (spec->n_det < 1 || spec->n_layers < 2 || spec->n_witness < 1) return fail(GW_EINVAL, "bad DeepClean spec");
    if (s->dc) return fail(GW_ESTATE, "stream already has a DeepClean stage");
    if (s->updates != 0) return fail(GW_ESTATE, "DeepClean must be created before the first update");
    if (spec->agg != GW_AGG_HANN_OLA && spec->agg != GW_AGG_LAST_STRIDE) return fail(GW_EINVAL, "unknown aggregation mode");
    if (spec->agg == GW_AGG_HANN_OLA && (s->W % s->S != 0 || s->W / s->S < 2))
        return fail(GW_EINVAL, "Hann overlap-add needs window %% stride == 0 and window/stride >= 2");
    if (spec->delta < 0 || spec->delta > s->W - s->S) return fail(GW_EINVAL, "delta out of range");
    for (int d = 0; d < spec->n_det; ++d) {
        if (spec->strain_row[d] < 0 || spec->strain_row[d] >= s->C) return fail(GW_EINVAL, "strain row out of range");
        for (int c = 0; c < spec->n_witness; ++c)
            if (spec->witness_rows[d * spec->n_witness + c] < 0 || spec->witness_rows[d * spec->n_witness + c] >= s->C)
                return fail(GW_EINVAL, "witness row out of range");
    }
    gw_options o;
    if (int rc = take_options(o, opts)) return rc;
    if (int rc = check_device()) return rc;
    gw_deepclean* dc = new gw_deepclean();
    dc->opt = o;
    dc->s = s; dc->n_det = spec->n_det; dc->n_layers = spec->n_layers; dc->n_wit = spec->n_witness;
    dc->agg = spec->agg; dc->delta = spec->delta;
    dc->fmt = dtype == GW_BF16 ? FMT_BF16 : FMT_FP16;
    int rc = deepclean_build(dc, s, spec);
    if (rc != GW_OK) { std::string keep = g_err; gw_deepclean_destroy(dc); g_err = keep; s->base.err = keep; return rc; }
    s->dc = dc;
    *out = dc;
    return GW_OK;
}

// a2, incremental: convert this update's S new witness samples into the mirror ring (after k_append).
static void ring16_append_enqueue(gw_deepclean* dc, const float* src, LaunchCtx& cx) {
    if (!dc->mirror) return;
    gw_stream* s = dc->s;
    cx.check(launch_ring16_append(src, dc->ring16, s->d_count, dc->d_rows_map, s->n, s->C, dc->n_det, dc->n_wit, s->W, s->S,
                                  dc->act_cols[0], dc->fmt, dc->d_pre, cx.next("ring16_append"), cx.st));
}

// `zones`: incremental handles only -- recompute the left-edge and right-edge rows of every layer (every update but the
// first, which fills the rings with whole windows).
static void deepclean_forward_enqueue(gw_deepclean* dc, LaunchCtx& cx, bool zones) {
    gw_stream* s = dc->s;
    if (!dc->mirror)
        cx.check(launch_gather(s->ring, dc->act[0], s->d_count, dc->d_rows_map, s->n, s->C, dc->n_det, dc->n_wit, s->W,
                               dc->act_cols[0], dc->fmt, dc->d_pre, cx.next("gather"), cx.st));
    size_t first = 0;
    if (dc->has_chain) { run_gemm(dc->chain, cx); first = 2; }    // layers 0 and 1 in one launch
    for (size_t i = first; i < dc->gemm.size(); ++i) run_gemm(dc->gemm[i], cx, zones && dc->inc);
    if (!dc->fused_tail)
        cx.check(launch_final_convt(dc->act[dc->n_layers - 1], dc->d_wt_final, dc->d_b_final, dc->pred, dc->batch, dc->n_det,
                                    dc->final_L, dc->final_cpad, dc->final_K, dc->final_pad, dc->fmt, cx.next("final_convt"), cx.st));
}

extern "C" int gw_deepclean_forward(gw_deepclean* dc, void* stream) {
    if (!dc) return fail(GW_EINVAL, "gw_deepclean_forward: NULL handle");
    CallScope scope(dc);
    if (dc->s->updates == 0 || dc->forward_for == dc->s->updates)
        return fail(GW_ESTATE, "gw_deepclean_forward: no new update to run on");
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    deepclean_forward_enqueue(dc, cx, dc->forward_for > 0);
    CX_TRY(cx, "gw_deepclean_forward");
    dc->forward_for = dc->s->updates;
    return GW_OK;
}

// ============================================================================ offline mode (D9)
struct gw_offline {
    HandleBase base;
    gw_stream* s = nullptr;                      // shape carrier only (n = windows per launch); no ring
    gw_deepclean* dc = nullptr;
    double* d_cum = nullptr;                     // [W] summed Hann weights along each residue chain
    int B = 0;
    long long T = 0;
};

extern "C" int gw_offline_destroy(gw_offline* o) {
    if (!o) return GW_OK;
    if (o->dc) { o->dc->s = nullptr; gw_deepclean_destroy(o->dc); }
    if (o->s) { cudaFree(o->s->d_count); cudaFree(o->s->d_ticket); delete o->s; }
    cudaFree(o->d_cum);
    o->base.magic = 0;
    delete o;
    return GW_OK;
}

extern "C" int gw_offline_create(gw_offline** out, const gw_dc_spec* spec, int channels, int fs, int window, int stride,
                                 int n_windows, int dtype, const gw_options* opts) {
    if (!out) return fail(GW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!spec || !spec->layers || !spec->witness_rows || !spec->strain_row) return fail(GW_EINVAL, "gw_offline_create: NULL argument");
    if (dtype != GW_BF16 && dtype != GW_FP16) return fail(GW_EINVAL, "dtype must be GW_BF16 or GW_FP16");
    if (channels < 1 || fs < 1 || window < 1 || stride < 1 || n_windows < 1) return fail(GW_EINVAL, "gw_offline_create: bad shape");
    if (window % stride != 0 || window / stride < 2) return fail(GW_EINVAL, "offline overlap-add needs window %% stride == 0 and window/stride >= 2");
    if (spec->n_det < 1 || spec->n_layers < 2 || spec->n_witness < 1) return fail(GW_EINVAL, "bad DeepClean spec");
    for (int d = 0; d < spec->n_det; ++d) {
        if (spec->strain_row[d] < 0 || spec->strain_row[d] >= channels) return fail(GW_EINVAL, "strain row out of range");
        for (int c = 0; c < spec->n_witness; ++c)
            if (spec->witness_rows[d * spec->n_witness + c] < 0 || spec->witness_rows[d * spec->n_witness + c] >= channels)
                return fail(GW_EINVAL, "witness row out of range");
    }
    gw_options oo;
    if (int rc = take_options(oo, opts)) return rc;
    if (oo.incremental) return fail(GW_EINVAL, "gw_offline_create: the incremental path is a streaming option");
    if (int rc = check_device()) return rc;
    gw_offline* o = new gw_offline();
    o->B = n_windows;
    o->T = static_cast<long long>(window) + static_cast<long long>(n_windows - 1) * stride;
    o->s = new gw_stream();
    o->s->n = n_windows; o->s->C = channels; o->s->fs = fs; o->s->W = window; o->s->S = stride;
    gw_deepclean* dc = new gw_deepclean();
    o->dc = dc;
    dc->opt = oo;
    dc->s = o->s; dc->n_det = spec->n_det; dc->n_layers = spec->n_layers; dc->n_wit = spec->n_witness;
    dc->agg = GW_AGG_HANN_OLA; dc->delta = 0; dc->offline = true; dc->off_T = o->T;
    dc->fmt = dtype == GW_BF16 ? FMT_BF16 : FMT_FP16;
    int rc = deepclean_build(dc, o->s, spec);
    if (rc == GW_OK) {
        std::vector<double> w(window), cum(window);
        const double pi = 3.14159265358979323846;
        for (int n = 0; n < window; ++n) w[n] = 0.5 - 0.5 * cos(2.0 * pi * n / window);
        for (int n = 0; n < window; ++n) {
            double sum = 0.0;
            for (int m = n; m < window; m += stride) sum += w[m];      // the order of the streaming path's table
            cum[n] = sum;
        }
        cudaError_t e = cudaMalloc(&o->d_cum, window * sizeof(double));
        if (e == cudaSuccess) e = cudaMemcpy(o->d_cum, cum.data(), window * sizeof(double), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) rc = fail(GW_ECUDA, "gw_offline_create: %s", cudaGetErrorString(e));
    }
    if (rc != GW_OK) { std::string keep = g_err; gw_offline_destroy(o); g_err = keep; return rc; }
    *out = o;
    return GW_OK;
}

extern "C" int gw_offline_set_scaling(gw_offline* o, const float* wit_mean, const float* wit_std, const float* strain_mean,
                                      const float* strain_std) {
    if (!o) return fail(GW_EINVAL, "gw_offline_set_scaling: NULL handle");
    CallScope scope(o);
    return set_scaling(o->dc, wit_mean, wit_std, strain_mean, strain_std);
}

extern "C" int64_t gw_offline_samples(const gw_offline* o) { return o ? o->T : 0; }

extern "C" int gw_offline_run(gw_offline* o, const float* samples_dev, float* cleaned_dev, float* noise_dev, void* stream) {
    if (!o || !samples_dev || !cleaned_dev) return fail(GW_EINVAL, "gw_offline_run: NULL argument");
    CallScope scope(o);
    gw_deepclean* dc = o->dc;
    gw_stream* s = o->s;
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    if (dc->seg16) {       // the whole segment as ONE "window" of length T: converts every sample once
        cx.check(launch_gather(samples_dev, dc->seg16, nullptr, dc->d_rows_map, 1, s->C, dc->n_det, dc->n_wit, static_cast<int>(o->T),
                               dc->act_cols[0], dc->fmt, dc->d_pre, nullptr, cx.st, o->T, 0));
    } else {
        cx.check(launch_gather(samples_dev, dc->act[0], nullptr, dc->d_rows_map, s->n, s->C, dc->n_det, dc->n_wit, s->W,
                               dc->act_cols[0], dc->fmt, dc->d_pre, nullptr, cx.st, o->T, s->S));
    }
    for (auto& g : dc->gemm) run_gemm(g, cx);
    if (!dc->fused_tail)
        cx.check(launch_final_convt(dc->act[dc->n_layers - 1], dc->d_wt_final, dc->d_b_final, dc->pred, dc->batch, dc->n_det,
                                    dc->final_L, dc->final_cpad, dc->final_K, dc->final_pad, dc->fmt, nullptr, cx.st));
    cx.check(launch_ola_offline(dc->pred, samples_dev, dc->d_strain_rows, dc->d_hann, o->d_cum, cleaned_dev, noise_dev, o->B,
                                dc->n_det, s->W, s->S, o->T, dc->d_post, cx.st));
    CX_TRY(cx, "gw_offline_run");
    dc->forward_for += 1;                        // gw_deepclean_noise-style hooks see a completed pass
    return GW_OK;
}

// Test hook: the raw per-window predictions [B][D][W] of the last gw_offline_run.
extern "C" int gw_offline_predictions(gw_offline* o, float* out_dev, void* stream) {
    if (!o || !out_dev) return fail(GW_EINVAL, "gw_offline_predictions: NULL argument");
    CallScope scope(o);
    CU_TRY(cudaMemcpyAsync(out_dev, o->dc->pred, static_cast<size_t>(o->dc->batch) * o->s->W * 4, cudaMemcpyDeviceToDevice,
                           static_cast<cudaStream_t>(stream)));
    return GW_OK;
}

// Time-ordered copy of a ring whose window starts at row h: dst[b][0 .. rows) = src[b][h .. h + rows) mod rows.
static int copy_unrotated(void* dst, const void* src, size_t row_bytes, size_t rows, size_t h, int batch, size_t src_rows,
                          cudaStream_t st) {
    const uint8_t* s8 = static_cast<const uint8_t*>(src);
    uint8_t* d8 = static_cast<uint8_t*>(dst);
    const size_t first = (h + rows <= src_rows) ? rows : src_rows - h;     // contiguous part
    CU_TRY(cudaMemcpy2DAsync(d8, rows * row_bytes, s8 + h * row_bytes, src_rows * row_bytes, first * row_bytes, batch,
                             cudaMemcpyDeviceToDevice, st));
    if (first < rows)
        CU_TRY(cudaMemcpy2DAsync(d8 + first * row_bytes, rows * row_bytes, s8, src_rows * row_bytes, (rows - first) * row_bytes,
                                 batch, cudaMemcpyDeviceToDevice, st));
    return GW_OK;
}

extern "C" int gw_deepclean_noise(gw_deepclean* dc, float* out_dev, void* stream) {
    if (!dc || !out_dev) return fail(GW_EINVAL, "gw_deepclean_noise: NULL argument");
    CallScope scope(dc);
    if (dc->forward_for == 0) return fail(GW_ESTATE, "gw_deepclean_noise: no forward pass yet");
    const size_t W = dc->s->W;
    if (dc->inc) {         // the prediction lives in a ring over absolute sample index: window position n is slot (count + n) mod W
        const size_t h = static_cast<size_t>((dc->forward_for * static_cast<int64_t>(dc->s->S)) % dc->s->W);
        return copy_unrotated(out_dev, dc->pred, 4, W, h, dc->batch, W, static_cast<cudaStream_t>(stream));
    }
    CU_TRY(cudaMemcpyAsync(out_dev, dc->pred, static_cast<size_t>(dc->batch) * W * 4, cudaMemcpyDeviceToDevice,
                           static_cast<cudaStream_t>(stream)));
    return GW_OK;
}

extern "C" int gw_deepclean_activation(gw_deepclean* dc, int layer, void* out_dev, int64_t out_bytes, int* rows,
                                       int* cols, void* stream) {
    if (!dc || layer < -1 || layer >= dc->n_layers - 1) return fail(GW_EINVAL, "gw_deepclean_activation: bad layer");
    CallScope scope(dc);
    const int i = layer + 1;
    if (i == dc->n_layers - 1 && dc->fused_tail && out_dev)
        return fail(GW_ESTATE, "layer %d's output is not materialised: it is fused with the final layer (gw_options.fuse_tail = 0 to inspect it)", layer);
    if (i == 1 && dc->has_chain && out_dev)
        return fail(GW_ESTATE, "layer 0's output is not materialised: layers 0 and 1 run as one kernel (gw_options.fuse_head = 0 to inspect it)");
    if (rows) *rows = dc->act_rows[i];
    if (cols) *cols = dc->act_cols[i];
    const int64_t bytes = static_cast<int64_t>(dc->batch) * dc->act_rows[i] * dc->act_cols[i] * 2;
    if (out_dev) {
        if (out_bytes < bytes) return fail(GW_EINVAL, "output buffer too small (%lld < %lld)", (long long)out_bytes, (long long)bytes);
        if ((i == 0 && dc->mirror) || (i > 0 && dc->inc)) {
            // the window is the contiguous row range [h_i, h_i + L_i) of each batch item's mirror ring (2 L_i rows)
            const size_t row_b = static_cast<size_t>(dc->act_cols[i]) * 2, L = dc->act_rows[i];
            const size_t hW = static_cast<size_t>((dc->s->updates * static_cast<int64_t>(dc->s->S)) % dc->s->W);
            const size_t h = hW / (static_cast<size_t>(dc->s->W) / L);
            const void* src = i == 0 ? dc->ring16 : dc->act[i];
            CU_TRY(cudaMemcpy2DAsync(out_dev, L * row_b, static_cast<const uint8_t*>(src) + h * row_b, 2 * L * row_b,
                                     L * row_b, dc->batch, cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(stream)));
        } else {
            CU_TRY(cudaMemcpyAsync(out_dev, dc->act[i], bytes, cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(stream)));
        }
    }
    return GW_OK;
}

static AggParams make_agg(gw_deepclean* dc, float* final_out, float* running_out, float* nhat_out) {
    gw_stream* s = dc->s;
    AggParams a;
    memset(&a, 0, sizeof a);
    a.pred = dc->pred; a.acc = dc->acc; a.ring = s->ring; a.count = s->d_count; a.strain_rows = dc->d_strain_rows;
    a.hann = dc->d_hann; a.inv_wsum = dc->d_inv_wsum; a.post = dc->d_post;
    a.final_out = final_out; a.running_out = running_out; a.nhat_out = nhat_out; a.clf_in = dc->clf_in;
    a.n_streams = s->n; a.n_det = dc->n_det; a.channels = s->C; a.W = s->W; a.S = s->S; a.Lb = dc->Lb;
    a.delta = dc->delta; a.agg = dc->agg;
    a.pred_ring = dc->inc ? 1 : 0;
    // the one-kernel classifier is one CTA of 288 threads per SM: as a programmatic dependent its prologue (barriers, TMEM,
    // weight loads) runs under this kernel's last wave without taking its thread slots
    a.trigger = (dc->bbh && dc->bbh->fused && dc->opt.pdl && dc->bbh->opt.pdl) ? 1 : 0;
    a.fir = dc->d_fir; a.hist = dc->d_hist; a.fir_n = dc->fir_n;
    return a;
}

static AggParams cleaned_enqueue(gw_deepclean* dc, float* final_out, float* running_out, float* nhat_out, LaunchCtx& cx) {
    AggParams a = make_agg(dc, final_out, running_out, nhat_out);
    a.stamp = cx.next("aggregate");
    cx.check(launch_aggregate(a, dc->opt.pdl, cx.st));
    return a;
}

extern "C" int gw_cleaned_strain(gw_deepclean* dc, float* out_dev, int mode, void* stream) {
    if (!dc) return fail(GW_EINVAL, "gw_cleaned_strain: NULL handle");
    CallScope scope(dc);
    if (mode != GW_FINAL && mode != GW_RUNNING) return fail(GW_EINVAL, "gw_cleaned_strain: bad mode");
    if (dc->forward_for != dc->s->updates || dc->cleaned_for == dc->s->updates)
        return fail(GW_ESTATE, "gw_cleaned_strain: call gw_deepclean_forward for this update first (once)");
    if (!dc->nhat) {
        const size_t wbytes = static_cast<size_t>(dc->batch) * dc->s->W * sizeof(float);
        CU_TRY(cudaMalloc(&dc->nhat, wbytes));
        CU_TRY(cudaMemset(dc->nhat, 0, wbytes));
    }
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    cleaned_enqueue(dc, mode == GW_FINAL ? out_dev : nullptr, mode == GW_RUNNING ? out_dev : nullptr, dc->nhat, cx);
    CX_TRY(cx, "gw_cleaned_strain");
    dc->cleaned_for = dc->s->updates;
    return GW_OK;
}

extern "C" int gw_noise_estimate(gw_deepclean* dc, float* out_dev, void* stream) {
    if (!dc || !out_dev) return fail(GW_EINVAL, "gw_noise_estimate: NULL argument");
    CallScope scope(dc);
    if (!dc->nhat || dc->cleaned_for == 0) return fail(GW_ESTATE, "gw_noise_estimate: call gw_cleaned_strain first");
    CU_TRY(cudaMemcpyAsync(out_dev, dc->nhat, static_cast<size_t>(dc->batch) * dc->s->W * 4, cudaMemcpyDeviceToDevice,
                           static_cast<cudaStream_t>(stream)));
    return GW_OK;
}

// ================================================================================ classifier
extern "C" int gw_bbh_destroy(gw_bbh* b) {
    if (!b) return GW_OK;
    for (auto& g : b->gemm) free_gemm(g);
    for (void* a : b->act) cudaFree(a);
    cudaFree(b->d_w1); cudaFree(b->d_b1); cudaFree(b->in_buf);
    cudaFree(b->d_hw1); cudaFree(b->d_hb1); cudaFree(b->d_hw2); cudaFree(b->d_hb2);
    cudaFree(b->pooled_dbg); cudaFree(b->scores_buf); cudaFree(b->d_whiten);
    cudaFree(b->d_w1img); cudaFree(b->d_w2img); cudaFree(b->d_w3img); cudaFree(b->d_fb1); cudaFree(b->d_fb2); cudaFree(b->d_fb3);
    if (b->dc && b->dc->bbh == b) { b->dc->bbh = nullptr; b->dc->clf_in = nullptr; b->dc->Lb = 0; }
    b->base.magic = 0;
    delete b;
    return GW_OK;
}

static int upload(float** dst, const float* src, size_t n) {
    CU_TRY(cudaMalloc(dst, n * 4));
    CU_TRY(cudaMemcpy(*dst, src, n * 4, cudaMemcpyHostToDevice));
    return GW_OK;
}

// One 16-bit value into a K-major SWIZZLE_128B operand image (rows of 128 bytes, 16-byte chunk c of row r at c ^ (r & 7)).
static void put_sw128(std::vector<uint16_t>& img, size_t block_elems, int row, int k, uint16_t bits) {
    img[block_elems + static_cast<size_t>(row) * 64 + (((k >> 3) ^ (row & 7)) << 3) + (k & 7)] = bits;
}

// gw_options.fuse_bbh: is this classifier one the one-kernel form takes (gw_bbh_fused.cu)?
static bool bbh_fused_shape(const std::vector<HostLayer>& H, int L, int hidden) {
    if (H.size() != 3) return false;
    for (const HostLayer& h : H)
        if (h.kind != GW_CONV || h.k != 8 || h.pad_l != 3 || h.stride != 1 || h.pool != 4) return false;
    return H[0].cout <= 32 && H[1].cin <= 32 && H[1].cout <= 64 && H[2].cin <= 64 && H[2].cout == 128 &&
           bbh_fused_supported(L, H[0].cin, hidden);
}

// Its operand images, host only (layouts: BbhFusedParams in gw_common.cuh).
static void bbh_fused_images(const std::vector<HostLayer>& H, int fmt, std::vector<uint16_t>& w1, std::vector<uint16_t>& w2,
                             std::vector<uint16_t>& w3) {
    const HostLayer &A = H[0], &B = H[1], &C = H[2];
    w1.assign(kBbhW1Bytes / 2, 0); w2.assign(kBbhW2Bytes / 2, 0); w3.assign(kBbhW3Bytes / 2, 0);
    // block 1: row n = phase q x 32 + cout, k = (cin x 2 + part) x 16 + i; input sample i of the row (position 4r - 3 + i)
    // is tap j = i - q of output phase q; the same weights multiply the hi and the lo part of a sample
    for (int q = 0; q < 4; ++q)
        for (int co = 0; co < A.cout; ++co)
            for (int ci = 0; ci < A.cin; ++ci)
                for (int j = 0; j < 8; ++j)
                    for (int part = 0; part < 2; ++part)
                        put_sw128(w1, 0, q * 32 + co, (ci * 2 + part) * 16 + j + q, to_storage_bits(A.W(co, ci, j), fmt));
    for (int j = 0; j < 8; ++j)
        for (int co = 0; co < B.cout; ++co)
            for (int ci = 0; ci < B.cin; ++ci)
                put_sw128(w2, static_cast<size_t>(j >> 1) * 64 * 64, co, (j & 1) * 32 + ci, to_storage_bits(B.W(co, ci, j), fmt));
    for (int j = 0; j < 8; ++j)
        for (int co = 0; co < C.cout; ++co)
            for (int ci = 0; ci < C.cin; ++ci)
                put_sw128(w3, static_cast<size_t>(j) * 128 * 64, co, ci, to_storage_bits(C.W(co, ci, j), fmt));
}

extern "C" int gw_bbh_fused_images(const gw_bbh_spec* spec, int dtype, uint16_t* w1, uint16_t* w2, uint16_t* w3) {
    if (!spec || !spec->convs || !spec->dense_dims || !w1 || !w2 || !w3) return fail(GW_EINVAL, "gw_bbh_fused_images: NULL argument");
    if (dtype != GW_BF16 && dtype != GW_FP16) return fail(GW_EINVAL, "dtype must be GW_BF16 or GW_FP16");
    if (spec->n_convs != 3 || spec->n_dense != 2) return fail(GW_EINVAL, "gw_bbh_fused_images: not a shape the one-kernel classifier takes");
    std::vector<HostLayer> H(3);
    for (int i = 0; i < 3; ++i)
        if (int rc = fold_layer(spec->convs[i], H[i])) return rc;
    if (!bbh_fused_shape(H, spec->length, spec->dense_dims[1])) return fail(GW_EINVAL, "gw_bbh_fused_images: not a shape the one-kernel classifier takes");
    std::vector<uint16_t> a, b, c;
    bbh_fused_images(H, dtype == GW_BF16 ? FMT_BF16 : FMT_FP16, a, b, c);
    memcpy(w1, a.data(), a.size() * 2); memcpy(w2, b.data(), b.size() * 2); memcpy(w3, c.data(), c.size() * 2);
    return GW_OK;
}

static int bbh_build_fused(gw_bbh* b, const std::vector<HostLayer>& H, int hidden) {
    const HostLayer &A = H[0], &B = H[1], &C = H[2];
    std::vector<uint16_t> w1, w2, w3;
    bbh_fused_images(H, b->fmt, w1, w2, w3);
    auto up16 = [](uint8_t** dst, const std::vector<uint16_t>& v) -> cudaError_t {
        cudaError_t e = cudaMalloc(dst, v.size() * 2);
        return e != cudaSuccess ? e : cudaMemcpy(*dst, v.data(), v.size() * 2, cudaMemcpyHostToDevice);
    };
    CU_TRY(up16(&b->d_w1img, w1));
    CU_TRY(up16(&b->d_w2img, w2));
    CU_TRY(up16(&b->d_w3img, w3));
    std::vector<float> b1(32, 0.f), b2(64, 0.f), b3(128, 0.f);
    for (int c = 0; c < A.cout; ++c) b1[c] = static_cast<float>(A.b[c]);
    for (int c = 0; c < B.cout; ++c) b2[c] = static_cast<float>(B.b[c]);
    for (int c = 0; c < C.cout; ++c) b3[c] = static_cast<float>(C.b[c]);
    if (int rc = upload(&b->d_fb1, b1.data(), 32)) return rc;
    if (int rc = upload(&b->d_fb2, b2.data(), 64)) return rc;
    if (int rc = upload(&b->d_fb3, b3.data(), 128)) return rc;
    b->hidden = hidden;
    CU_TRY(bbh_fused_prepare());
    b->fused = true;
    return GW_OK;
}

static int bbh_build(gw_bbh* b, const gw_bbh_spec* spec) {
    const int nc = spec->n_convs;
    std::vector<HostLayer> H(nc);
    int L = spec->length;
    for (int i = 0; i < nc; ++i) {
        if (int rc = fold_layer(spec->convs[i], H[i])) return rc;
        if (H[i].kind != GW_CONV || H[i].stride != 1 || H[i].pad_l + H[i].pad_r != H[i].k - 1 || H[i].pool != 4 ||
            H[i].act != GW_ACT_RELU)
            return fail(GW_EINVAL, "classifier blocks must be Conv1d stride 1 'same' padding + ReLU + MaxPool(4)");
        if (i > 0 && H[i].cin != H[i - 1].cout) return fail(GW_EINVAL, "classifier block %d cin mismatch", i);
    }
    if (H[0].cin != b->n_det) return fail(GW_EINVAL, "first classifier block cin must equal the number of detectors");
    if (spec->n_dense != 2 || spec->dense_dims[0] != H[nc - 1].cout || spec->dense_dims[2] != 1)
        return fail(GW_EINVAL, "dense head must be cout -> hidden -> 1");
    const int hidden = spec->dense_dims[1];
    if (hidden < 1 || hidden > 128) return fail(GW_EINVAL, "dense hidden width must be in [1,128]");
    CU_TRY(cudaMalloc(&b->in_buf, static_cast<size_t>(b->batch) * b->n_det * L * 4));
    CU_TRY(cudaMemset(b->in_buf, 0, static_cast<size_t>(b->batch) * b->n_det * L * 4));
    CU_TRY(cudaMalloc(&b->scores_buf, static_cast<size_t>(b->batch) * 4));
    if (int rc = upload(&b->d_hw1, spec->dense_w[0], static_cast<size_t>(hidden) * spec->dense_dims[0])) return rc;
    if (int rc = upload(&b->d_hb1, spec->dense_b[0], hidden)) return rc;
    if (int rc = upload(&b->d_hw2, spec->dense_w[1], hidden)) return rc;
    if (int rc = upload(&b->d_hb2, spec->dense_b[1], 1)) return rc;
    {
        int l = L;
        for (int i = 0; i < nc; ++i) { b->flops += 2.0 * l * H[i].k * H[i].cin * H[i].cout; l /= 4; }
    }
    // the whole classifier as one kernel when its shape is the one that kernel is written for (BASELINE.json configs[2])
    if (b->opt.fuse_bbh && b->opt.conv_impl == GW_IMPL_UMMA && bbh_fused_shape(H, L, hidden)) return bbh_build_fused(b, H, hidden);
    // first block on CUDA cores (its cin * k taps live in registers)
    if (H[0].cin > 4 || H[0].k > 8 || H[0].pad_l > 4 || H[0].k - 1 - H[0].pad_l > 4)
        return fail(GW_EINVAL, "first classifier block: needs cin <= 4, k <= 8, pad_l <= 4, pad_r <= 4");
    b->c1 = H[0];
    b->c1_cpad = round_up(H[0].cout, 32);
    {
        std::vector<float> w(H[0].w.size()), bb(H[0].cout);
        for (size_t i = 0; i < w.size(); ++i) w[i] = static_cast<float>(storage_to_double(to_storage_bits(H[0].w[i], b->fmt), b->fmt));
        for (int c = 0; c < H[0].cout; ++c) bb[c] = static_cast<float>(H[0].b[c]);
        if (int rc = upload(&b->d_w1, w.data(), w.size())) return rc;
        if (int rc = upload(&b->d_b1, bb.data(), bb.size())) return rc;
    }
    // activations: act[i] = input of block i+1 = pooled output of block i
    b->act.assign(nc - 1, nullptr);
    std::vector<int> len(nc), cp(nc);
    int l = L;
    for (int i = 0; i < nc - 1; ++i) {
        l /= 4;
        len[i] = l; cp[i] = round_up(H[i].cout, 32);
        CU_TRY(cudaMalloc(&b->act[i], static_cast<size_t>(b->batch) * l * cp[i] * 2));
        CU_TRY(cudaMemset(b->act[i], 0, static_cast<size_t>(b->batch) * l * cp[i] * 2));
    }
    b->gemm.resize(nc - 1);
    for (int i = 1; i < nc; ++i) {
        const bool last = i == nc - 1;
        const int cout_p = round_up(H[i].cout, 32);
        if (last && len[i - 1] / 2 > kTileM) return fail(GW_EINVAL, "classifier window too long for the fused head");
        if (last && cout_p != H[i].cout) return fail(GW_EINVAL, "last classifier block cout must be a multiple of 32");
        if (len[i - 1] % 4) return fail(GW_EINVAL, "classifier length must be divisible by 4^blocks");
        GemmLayer& gl = b->gemm[i - 1];
        if (int rc = build_gemm_layer(gl, GK_BBH, &H[i], 1, b->fmt, b->opt, b->act[i - 1], len[i - 1], cp[i - 1],
                                      last ? nullptr : b->act[i], cout_p, b->batch, last ? EPI_POOL_HEAD : EPI_POOL,
                                      last ? hidden : 0))
            return rc;
        gl.name = "gemm.bbh" + std::to_string(i);
        gl.flops = 2.0 * len[i - 1] * H[i].k * H[i].cin * H[i].cout;
        if (last) {
            ConvGemmParams& p = gl.g.p;
            p.hw1 = b->d_hw1; p.hb1 = b->d_hb1; p.hw2 = b->d_hw2; p.hb2 = b->d_hb2; p.head_hidden = hidden;
            p.scores = b->scores_buf;
            CU_TRY(cudaMalloc(&b->pooled_dbg, static_cast<size_t>(b->batch) * (p.M / 2) * (p.N / 2) * 4));
            p.pooled_dbg = b->pooled_dbg;
        }
    }
    CU_TRY(conv_gemm_prepare());
    return GW_OK;
}

extern "C" int gw_bbh_create(gw_bbh** out, gw_deepclean* dc, const gw_bbh_spec* spec, int dtype, int n_det, int max_batch,
                             const gw_options* opts) {
    if (!out) return fail(GW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!spec || !spec->convs || !spec->dense_dims || !spec->dense_w || !spec->dense_b) return fail(GW_EINVAL, "gw_bbh_create: NULL argument");
    CallScope scope(dc);
    if (dtype != GW_BF16 && dtype != GW_FP16) return fail(GW_EINVAL, "dtype must be GW_BF16 or GW_FP16");
    if (spec->n_convs < 2) return fail(GW_EINVAL, "classifier needs at least 2 conv blocks");
    if (spec->length < 64 || spec->length % 64) return fail(GW_EINVAL, "classifier length must be a multiple of 64");
    if (dc) {
        if (dc->bbh) return fail(GW_ESTATE, "DeepClean stage already has a classifier");
        if (spec->length + dc->delta > dc->s->W) return fail(GW_EINVAL, "classifier window + delta exceeds the snapshot window");
        n_det = dc->n_det; max_batch = dc->s->n;
    } else if (n_det < 1 || max_batch < 1) {
        return fail(GW_EINVAL, "stateless classifier needs n_det >= 1 and max_batch >= 1");
    }
    gw_options o;
    if (int rc = take_options(o, opts)) return rc;
    o.incremental = 0;                           // a DeepClean option; the classifier window is rescored every update
    if (int rc = check_device()) return rc;
    gw_bbh* b = new gw_bbh();
    b->opt = o;
    b->dc = dc; b->n_det = n_det; b->batch = max_batch; b->L = spec->length;
    b->fmt = dtype == GW_BF16 ? FMT_BF16 : FMT_FP16;
    int rc = bbh_build(b, spec);
    if (rc != GW_OK) { std::string keep = g_err; b->dc = nullptr; gw_bbh_destroy(b); g_err = keep; if (dc) dc->base.err = keep; return rc; }
    if (dc) { dc->bbh = b; dc->clf_in = b->in_buf; dc->Lb = b->L; }
    *out = b;
    return GW_OK;
}

// D12: causal FIR whitening of every detector's classifier window, zero initial state.
extern "C" int gw_bbh_set_whitening(gw_bbh* b, const float* taps_host, int n_taps) {
    if (!b) return fail(GW_EINVAL, "gw_bbh_set_whitening: NULL handle");
    CallScope scope(b);
    cudaFree(b->d_whiten);
    b->d_whiten = nullptr; b->whiten_n = 0;
    if (!taps_host || n_taps == 0) return GW_OK;
    if (n_taps < 1 || n_taps > kMaxFir) return fail(GW_EINVAL, "whitening needs 1 <= n_taps <= %d", kMaxFir);
    const size_t n = static_cast<size_t>(b->n_det) * n_taps;
    for (size_t i = 0; i < n; ++i)
        if (!isfinite(taps_host[i])) return fail(GW_EINVAL, "whitening taps must be finite");
    CU_TRY(cudaMalloc(&b->d_whiten, n * sizeof(float)));
    CU_TRY(cudaMemcpy(b->d_whiten, taps_host, n * sizeof(float), cudaMemcpyHostToDevice));
    b->whiten_n = n_taps;
    return GW_OK;
}

static void bbh_enqueue(gw_bbh* b, const float* in, int batch, LaunchCtx& cx) {
    if (b->fused) {
        BbhFusedParams q = {};
        q.x = in; q.w1img = b->d_w1img; q.w2img = b->d_w2img; q.w3img = b->d_w3img;
        q.b1 = b->d_fb1; q.b2 = b->d_fb2; q.b3 = b->d_fb3;
        q.hw1 = b->d_hw1; q.hb1 = b->d_hb1; q.hw2 = b->d_hw2; q.hb2 = b->d_hb2;
        q.whiten = b->d_whiten; q.whiten_n = b->whiten_n;
        q.scores = b->scores_buf;
        q.L = b->L; q.cin = b->n_det; q.hidden = b->hidden;
        q.stamp = cx.next("bbh_fused", b->flops * batch);
        cx.check(launch_bbh_fused(q, batch, b->fmt, b->opt.pdl, cx.st));
        return;
    }
    cx.check(launch_bbh_conv1(in, b->d_w1, b->d_b1, b->act[0], batch, b->n_det, b->L, b->c1.cout, b->c1_cpad, b->c1.k,
                              b->c1.pad_l, b->c1.pool, b->fmt, b->d_whiten, b->whiten_n, b->opt.pdl, cx.next("bbh_conv1"), cx.st));
    for (auto& g : b->gemm) run_gemm(g, cx, false, batch);
}

extern "C" int gw_bbh_score(gw_bbh* b, float* scores_dev, void* stream) {
    if (!b || !scores_dev) return fail(GW_EINVAL, "gw_bbh_score: NULL argument");
    CallScope scope(b);
    if (!b->dc) return fail(GW_ESTATE, "gw_bbh_score: stateless classifier; use gw_bbh_score_batch");
    if (b->dc->cleaned_for != b->dc->s->updates || b->dc->cleaned_for == 0 || b->scored_for == b->dc->s->updates)
        return fail(GW_ESTATE, "gw_bbh_score: call gw_cleaned_strain for this update first (once)");
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    bbh_enqueue(b, b->in_buf, b->batch, cx);
    CX_TRY(cx, "gw_bbh_score");
    CU_TRY(cudaMemcpyAsync(scores_dev, b->scores_buf, static_cast<size_t>(b->batch) * 4, cudaMemcpyDeviceToDevice, cx.st));
    b->scored_for = b->dc->s->updates;
    return GW_OK;
}

extern "C" int gw_bbh_score_batch(gw_bbh* b, const float* windows_dev, int batch, float* scores_dev, void* stream) {
    if (!b || !windows_dev || !scores_dev) return fail(GW_EINVAL, "gw_bbh_score_batch: NULL argument");
    CallScope scope(b);
    if (batch < 1 || batch > b->batch) return fail(GW_EINVAL, "batch %d outside [1, %d]", batch, b->batch);
    LaunchCtx cx(static_cast<cudaStream_t>(stream));
    bbh_enqueue(b, windows_dev, batch, cx);
    CX_TRY(cx, "gw_bbh_score_batch");
    CU_TRY(cudaMemcpyAsync(scores_dev, b->scores_buf, static_cast<size_t>(batch) * 4, cudaMemcpyDeviceToDevice, cx.st));
    return GW_OK;
}

// ================================================================================== pipeline
extern "C" int gw_pipeline_create(gw_pipeline** out, gw_stream* s, gw_deepclean* dc, gw_bbh* bbh) {
    if (!out) return fail(GW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!s || !dc || dc->s != s || (bbh && bbh->dc != dc)) return fail(GW_EINVAL, "gw_pipeline_create: stages do not belong together");
    gw_pipeline* p = new gw_pipeline();
    p->s = s; p->dc = dc; p->bbh = bbh;
    *out = p;
    return GW_OK;
}

static void graphvar_reset(GraphVar& v) {
    if (v.exec) cudaGraphExecDestroy(v.exec);
    if (v.graph) cudaGraphDestroy(v.graph);
    v = GraphVar();
}

extern "C" int gw_pipeline_destroy(gw_pipeline* p) {
    if (!p) return GW_OK;
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) graphvar_reset(p->var[a][b]);
    cudaFree(p->d_stamps);
    cudaFree(p->d_in); cudaFree(p->d_scores); cudaFree(p->d_final);
    for (int i = 0; i < 2; ++i) {
        cudaFree(p->d_in2[i]);
        if (p->in_done[i]) cudaEventDestroy(p->in_done[i]);
        if (p->in_free[i]) cudaEventDestroy(p->in_free[i]);
    }
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    p->base.magic = 0;
    delete p;
    return GW_OK;
}

// Kernel nodes of the graph the steps replay (the non-profiling variant; incremental handles: the zones variant once
// it exists).  0 before the first gw_step.
extern "C" int gw_pipeline_graph_nodes(const gw_pipeline* p) {
    if (!p) return 0;
    if (p->var[1][0].exec) return p->var[1][0].nodes;
    return p->var[0][0].nodes;
}

// Capture update -> forward -> cleaned(GW_FINAL) -> score into `v`.  zones: incremental handles after their first
// update; stamped: every kernel also records its %globaltimer span (gw_step_profile).
static int pipeline_capture(gw_pipeline* p, GraphVar& v, bool zones, bool stamped, const float* in, float* scores, float* fin,
                            cudaStream_t st) {
    graphvar_reset(v);
    LaunchCtx cx(st);
    if (stamped) {
        if (!p->d_stamps) CU_TRY(cudaMalloc(&p->d_stamps, kMaxStamps * kStampSlots * sizeof(unsigned long long)));
        cx.stamps = p->d_stamps;
        cx.prof = &v.prof;
    }
    const long long before = kernel_launches();
    CU_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    if (stamped) cx.check(launch_stamp_init(p->d_stamps, kMaxStamps, st));
    stream_update_enqueue(p->s, in, cx);
    deepclean_forward_enqueue(p->dc, cx, zones);
    v.agg = cleaned_enqueue(p->dc, fin, nullptr, nullptr, cx);
    if (p->bbh) {
        bbh_enqueue(p->bbh, p->bbh->in_buf, p->bbh->batch, cx);
        // cudaMemcpyDefault: `scores` may be the device alias of a pinned host buffer (gw_step_host_async)
        cx.check(cudaMemcpyAsync(scores, p->bbh->scores_buf, static_cast<size_t>(p->bbh->batch) * 4, cudaMemcpyDefault, st));
    }
    cudaError_t e = cudaStreamEndCapture(st, &v.graph);
    const long long captured = kernel_launches() - before;
    uncount_launches(captured);                         // captured, not launched
    v.nodes = static_cast<int>(captured);
    if (cx.err != cudaSuccess || e != cudaSuccess) {
        const cudaError_t shown = cx.err != cudaSuccess ? cx.err : e;
        if (v.graph) { cudaGraphDestroy(v.graph); v.graph = nullptr; }
        cudaGetLastError();
        return fail(GW_ECUDA, "graph capture failed: %s", cudaGetErrorString(shown));
    }
    CU_TRY(cudaGraphInstantiate(&v.exec, v.graph, 0));
    v.cap_in = in; v.cap_scores = scores; v.cap_final = fin;
    // remember the nodes that hold caller pointers: new buffers are then parameter updates, not re-captures
    size_t n_nodes = 0;
    CU_TRY(cudaGraphGetNodes(v.graph, nullptr, &n_nodes));
    std::vector<cudaGraphNode_t> nodes(n_nodes);
    CU_TRY(cudaGraphGetNodes(v.graph, nodes.data(), &n_nodes));
    for (cudaGraphNode_t nd : nodes) {
        cudaGraphNodeType ty;
        CU_TRY(cudaGraphNodeGetType(nd, &ty));
        if (ty == cudaGraphNodeTypeMemcpy) { v.scores_node = nd; continue; }
        if (ty != cudaGraphNodeTypeKernel) continue;
        cudaKernelNodeParams kp;
        CU_TRY(cudaGraphKernelNodeGetParams(nd, &kp));
        if (is_append_kernel(kp.func)) { v.append_node = nd; v.append_fused = false; }
        if (is_snapshot_append_kernel(kp.func)) { v.append_node = nd; v.append_fused = true; }
        if (is_ring16_append_kernel(kp.func)) v.ring16_node = nd;
        if (is_aggregate_kernel(kp.func)) v.agg_node = nd;
    }
    return GW_OK;
}

// Replace argument `idx` of a kernel node of the instantiated graph (the other n_args - 1 arguments are kept).
static int set_kernel_arg(GraphVar& v, cudaGraphNode_t node, int n_args, int idx, void* value) {
    cudaKernelNodeParams kp;
    CU_TRY(cudaGraphKernelNodeGetParams(node, &kp));
    void* args[20];
    for (int i = 0; i < n_args; ++i) args[i] = kp.kernelParams[i];
    args[idx] = value;
    kp.kernelParams = args;
    CU_TRY(cudaGraphExecKernelNodeSetParams(v.exec, node, &kp));
    CU_TRY(cudaGraphKernelNodeSetParams(node, &kp));    // keep the template graph in step (later Get/Set pairs start from it)
    return GW_OK;
}

static int pipeline_set_input(GraphVar& v, const float* in) {
    // k_append(ring, src, count, ticket, n_rows, W, S, stamp); k_ring16_append(src, ring16, count, rows_map, ... 13 args)
    // k_snapshot_append(ring, src, ring16, count, ticket, rows_map, pre, ... 15 args)
    const float* src = in;
    if (v.append_fused) {
        if (int rc = set_kernel_arg(v, v.append_node, 15, 1, &src)) return rc;
    } else {
        if (int rc = set_kernel_arg(v, v.append_node, 8, 1, &src)) return rc;
        if (v.ring16_node)
            if (int rc = set_kernel_arg(v, v.ring16_node, 13, 0, &src)) return rc;
    }
    v.cap_in = in;
    return GW_OK;
}

// One update through the graph variant that applies; captures it on first use, otherwise patches the node parameters
// that hold caller pointers.  *used receives the variant (gw_step_profile reads its stamps).
static int pipeline_run(gw_pipeline* p, const float* in, float* scores, float* fin, cudaStream_t st, bool stamped,
                        GraphVar** used) {
    const bool zones = p->dc->inc && p->s->updates > 0;
    GraphVar& v = p->var[zones ? 1 : 0][stamped ? 1 : 0];
    bool capture = !v.exec || (v.cap_in != in && !v.append_node) || (v.cap_final != fin && !v.agg_node) ||
                   (p->bbh && v.cap_scores != scores && !v.scores_node);
    if (!capture) {
        if (v.cap_in != in)
            if (int rc = pipeline_set_input(v, in)) return rc;
        if (v.cap_final != fin) {
            AggParams a = v.agg;
            a.final_out = fin;
            if (int rc = set_kernel_arg(v, v.agg_node, 1, 0, &a)) return rc;
            v.agg = a; v.cap_final = fin;
        }
        if (p->bbh && v.cap_scores != scores) {
            const size_t bytes = static_cast<size_t>(p->bbh->batch) * 4;
            cudaError_t e = cudaGraphExecMemcpyNodeSetParams1D(v.exec, v.scores_node, scores, p->bbh->scores_buf, bytes, cudaMemcpyDefault);
            if (e == cudaSuccess) e = cudaGraphMemcpyNodeSetParams1D(v.scores_node, scores, p->bbh->scores_buf, bytes, cudaMemcpyDefault);
            if (e == cudaSuccess) v.cap_scores = scores;
            else { cudaGetLastError(); capture = true; }    // e.g. device buffer -> mapped host buffer: a different copy kind
        }
    }
    if (capture) {
        if (st == nullptr) return fail(GW_EINVAL, "gw_step needs a non-default stream (graph capture)");
        if (int rc = pipeline_capture(p, v, zones, stamped, in, scores, fin, st)) return rc;
    }
    CU_TRY(cudaGraphLaunch(v.exec, st));
    for (int i = 0; i < v.nodes; ++i) count_launch();
    p->s->updates += 1;
    p->dc->forward_for = p->dc->cleaned_for = p->s->updates;
    if (p->bbh) p->bbh->scored_for = p->s->updates;
    if (used) *used = &v;
    return GW_OK;
}

extern "C" int gw_step(gw_pipeline* p, const float* new_samples_dev, float* scores_dev, float* cleaned_final_dev, void* stream) {
    if (!p || !new_samples_dev || !cleaned_final_dev || (p->bbh && !scores_dev)) return fail(GW_EINVAL, "gw_step: NULL argument");
    CallScope scope(p);
    if (int rc = stream_update_checked(p->s)) return rc;
    return pipeline_run(p, new_samples_dev, scores_dev, cleaned_final_dev, static_cast<cudaStream_t>(stream), false, nullptr);
}

// One update through the PROFILING graph: the same kernels and launch attributes as gw_step, each stamping
// %globaltimer at its first CTA's start and its last CTA's end; synchronises.
extern "C" int gw_step_profile(gw_pipeline* p, const float* new_samples_dev, float* scores_dev, float* cleaned_final_dev,
                               void* stream, int max_kernels, double* begin_us, double* end_us, double* sm_mhz, int* n_out) {
    if (!p || !new_samples_dev || !cleaned_final_dev || !begin_us || !end_us || !n_out || (p->bbh && !scores_dev))
        return fail(GW_EINVAL, "gw_step_profile: NULL argument");
    CallScope scope(p);
    if (int rc = stream_update_checked(p->s)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    GraphVar* v = nullptr;
    if (int rc = pipeline_run(p, new_samples_dev, scores_dev, cleaned_final_dev, st, true, &v)) return rc;
    CU_TRY(cudaStreamSynchronize(st));
#ifdef GW_TRACE
    for (auto& g : p->dc->gemm) trace_report(g);
    if (p->bbh) for (auto& g : p->bbh->gemm) trace_report(g);
#endif
    unsigned long long h[kMaxStamps * kStampSlots];
    CU_TRY(cudaMemcpy(h, p->d_stamps, sizeof h, cudaMemcpyDeviceToHost));
    const int nk = static_cast<int>(v->prof.labels.size());
    unsigned long long t0 = ~0ull;
    for (int i = 0; i < nk; ++i) if (h[kStampSlots * i] < t0) t0 = h[kStampSlots * i];
    *n_out = nk;
    for (int i = 0; i < nk && i < max_kernels; ++i) {
        const unsigned long long* s = h + kStampSlots * i;
        begin_us[i] = static_cast<double>(s[0] - t0) * 1e-3;
        end_us[i] = static_cast<double>(s[1] - t0) * 1e-3;
        if (sm_mhz) sm_mhz[i] = s[5] > s[4] ? static_cast<double>(s[3] - s[2]) / static_cast<double>(s[5] - s[4]) * 1e3 : 0.0;
    }
    p->last_prof = &v->prof;
    return GW_OK;
}

extern "C" const char* gw_profile_label(const gw_pipeline* p, int i) {
    if (!p || !p->last_prof || i < 0 || i >= static_cast<int>(p->last_prof->labels.size())) return "";
    return p->last_prof->labels[i].c_str();
}
extern "C" double gw_profile_flops(const gw_pipeline* p, int i) {
    if (!p || !p->last_prof || i < 0 || i >= static_cast<int>(p->last_prof->flops.size())) return 0.0;
    return p->last_prof->flops[i];
}
extern "C" double gw_profile_smem_bytes(const gw_pipeline* p, int i) {
    if (!p || !p->last_prof || i < 0 || i >= static_cast<int>(p->last_prof->smem.size())) return 0.0;
    return p->last_prof->smem[i];
}

// Throughput form of gw_step_host: does NOT synchronise, and the host->device copy of this call's samples
// runs on an internal copy stream into one of two staging buffers, so it overlaps the previous step's kernels
// (at C4 n=128 the copy is 11.5 MB, about a quarter of the step).  Results land in the host buffers in stream
// order on `stream`; all host buffers of a call must stay valid until `stream` has been synchronised past it.
extern "C" int gw_step_host_async(gw_pipeline* p, const float* new_samples_host, float* scores_host,
                                  float* cleaned_final_host, void* stream) {
    if (!p || !new_samples_host || !cleaned_final_host || (p->bbh && !scores_host))
        return fail(GW_EINVAL, "gw_step_host_async: NULL argument");
    CallScope scope(p);
    gw_stream* s = p->s;
    if (int rc = stream_update_checked(s)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t in_bytes = static_cast<size_t>(s->n) * s->C * s->S * 4;
    const size_t fin_bytes = static_cast<size_t>(p->dc->batch) * s->S * 4;
    const size_t sc_bytes = static_cast<size_t>(s->n) * 4;
    if (!p->copy_stream) {
        CU_TRY(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CU_TRY(cudaMalloc(&p->d_in2[i], in_bytes));
            CU_TRY(cudaEventCreateWithFlags(&p->in_done[i], cudaEventDisableTiming));
            CU_TRY(cudaEventCreateWithFlags(&p->in_free[i], cudaEventDisableTiming));
        }
    }
    if (!p->d_final) CU_TRY(cudaMalloc(&p->d_final, fin_bytes));
    if (!p->d_scores) CU_TRY(cudaMalloc(&p->d_scores, sc_bytes));
    const int b = static_cast<int>(p->async_calls & 1);
    if (p->async_calls >= 2) CU_TRY(cudaStreamWaitEvent(p->copy_stream, p->in_free[b], 0));   // step k-2 has read it
    CU_TRY(cudaMemcpyAsync(p->d_in2[b], new_samples_host, in_bytes, cudaMemcpyHostToDevice, p->copy_stream));
    CU_TRY(cudaEventRecord(p->in_done[b], p->copy_stream));
    CU_TRY(cudaStreamWaitEvent(st, p->in_done[b], 0));
    // Pinned (mapped) host output buffers are written by the kernels themselves -- 0.5 MB of posted PCIe writes from
    // the overlap-add kernel and n scores from the classifier head -- instead of by two copies behind the graph.
    void *fin_alias = nullptr, *sc_alias = nullptr;
    const bool direct = cudaHostGetDevicePointer(&fin_alias, cleaned_final_host, 0) == cudaSuccess &&
                        (!p->bbh || cudaHostGetDevicePointer(&sc_alias, scores_host, 0) == cudaSuccess);
    if (!direct) cudaGetLastError();             // pageable memory: clear the sticky-free error, use the copies
    if (direct) {
        if (int rc = pipeline_run(p, p->d_in2[b], p->bbh ? static_cast<float*>(sc_alias) : p->d_scores,
                                  static_cast<float*>(fin_alias), st, false, nullptr)) return rc;
        CU_TRY(cudaEventRecord(p->in_free[b], st));
    } else {
        if (int rc = pipeline_run(p, p->d_in2[b], p->d_scores, p->d_final, st, false, nullptr)) return rc;
        CU_TRY(cudaEventRecord(p->in_free[b], st));
        CU_TRY(cudaMemcpyAsync(cleaned_final_host, p->d_final, fin_bytes, cudaMemcpyDeviceToHost, st));
        if (p->bbh) CU_TRY(cudaMemcpyAsync(scores_host, p->d_scores, sc_bytes, cudaMemcpyDeviceToHost, st));
    }
    p->async_calls += 1;
    return GW_OK;
}

extern "C" int gw_step_host(gw_pipeline* p, const float* new_samples_host, float* scores_host, float* cleaned_final_host, void* stream) {
    if (!p || !new_samples_host || !cleaned_final_host || (p->bbh && !scores_host)) return fail(GW_EINVAL, "gw_step_host: NULL argument");
    CallScope scope(p);
    gw_stream* s = p->s;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t in_bytes = static_cast<size_t>(s->n) * s->C * s->S * 4;
    const size_t fin_bytes = static_cast<size_t>(p->dc->batch) * s->S * 4;
    const size_t sc_bytes = static_cast<size_t>(s->n) * 4;
    if (!p->d_in) CU_TRY(cudaMalloc(&p->d_in, in_bytes));
    if (!p->d_final) CU_TRY(cudaMalloc(&p->d_final, fin_bytes));
    if (!p->d_scores) CU_TRY(cudaMalloc(&p->d_scores, sc_bytes));
    if (int rc = stream_update_checked(s)) return rc;
    CU_TRY(cudaMemcpyAsync(p->d_in, new_samples_host, in_bytes, cudaMemcpyHostToDevice, st));
    if (int rc = pipeline_run(p, p->d_in, p->d_scores, p->d_final, st, false, nullptr)) return rc;
    CU_TRY(cudaMemcpyAsync(cleaned_final_host, p->d_final, fin_bytes, cudaMemcpyDeviceToHost, st));
    if (p->bbh) CU_TRY(cudaMemcpyAsync(scores_host, p->d_scores, sc_bytes, cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    return GW_OK;
}
