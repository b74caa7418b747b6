/*
 * gw_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the hot path of arXiv:2108.12430
 * computes (snapshotter -> DeepClean-style conv autoencoder -> Hann overlap-add + subtraction
 * -> BBH 1-D CNN classifier).  Every function is the textbook definition written out as nested
 * loops, in the notation of DESIGN.md section "Definitions" (D1..D8), each citing the passage of
 * /root/reference/PAPER.md (or the BASELINE.json config) it follows.  No blocking, no fusion, no
 * reordering, no intrinsics.  The only concession to run time is one OpenMP `parallel for` on
 * the outermost (output-channel) loop of the two convolutions; it does not change any sum.
 *
 * It shares no code with the CUDA path (paper_2108_12430_b200/csrc) and neither includes
 * the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py against something
 * other than itself (impulse responses, adjoint identity, closed forms, brute force, the
 * float64 routines of a library); see the table in DESIGN.md.  Nothing here is "parity unpinned".
 * The paper prints no numeric worked example for any stage (all figures are images), so there
 * are no paper-printed golden values to check; DESIGN.md says so.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int gwo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void gwo_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * D1  Snapshot (B.1: "a state representing the previous input snapshot ... a
 * floor(fs/r)-sized stream of strictly new samples that are used to update the state to a new
 * snapshot").  x_c[a] is channel c's sample with absolute index a >= 0, x_c[a] = 0 for a < 0
 * (reading A12: the state starts as zeros).  After update t (t = 0,1,...):
 *     snapshot_t[c][n] = x_c[(t+1)*S - W + n],  n in [0, W).
 * x: [C][T] float (all samples so far, T >= (t+1)*S).  out: [C][W].  Samples are moved, never
 * computed on, so this is float32 in / float32 out and bit-exact by definition.
 * -------------------------------------------------------------------------------------------*/
void gwo_snapshot(const float *x, int C, int64_t T, int64_t t, int S, int W, float *out,
                  int64_t *first_index) {
    int64_t first = (t + 1) * (int64_t)S - W;
    for (int c = 0; c < C; ++c) {
        for (int n = 0; n < W; ++n) {
            int64_t a = first + n;
            out[(int64_t)c * W + n] = (a < 0) ? 0.0f : x[(int64_t)c * T + a];
        }
    }
    *first_index = first;
}

/* ---------------------------------------------------------------------------------------------
 * D2  Conv1d (cross-correlation; the layer type BASELINE.json configs[0..2] name; DeepClean is
 * "a 1-D convolutional autoencoder"; BBHnet "1-D convolutional neural networks",
 * PAPER.md:38):
 *     y[co][l] = b[co] + sum_ci sum_{j=0}^{K-1} w[co][ci][j] * xt[ci][s*l + j - pL],
 *     xt = x inside [0, L), 0 outside;  L_out = floor((L + pL + pR - K)/s) + 1.
 * x: [Cin][L], w: [Cout][Cin][K], y: [Cout][L_out].
 * -------------------------------------------------------------------------------------------*/
int gwo_conv1d_lout(int L, int K, int s, int pL, int pR) { return (L + pL + pR - K) / s + 1; }

void gwo_conv1d(const double *x, const double *w, const double *b, int Cin, int Cout, int L, int K,
                int s, int pL, int pR, double *y) {
    int Lout = gwo_conv1d_lout(L, K, s, pL, pR);
#pragma omp parallel for schedule(static)
    for (int co = 0; co < Cout; ++co) {
        for (int l = 0; l < Lout; ++l) {
            double acc = b ? b[co] : 0.0;
            for (int ci = 0; ci < Cin; ++ci) {
                for (int j = 0; j < K; ++j) {
                    int i = s * l + j - pL;
                    if (i >= 0 && i < L)
                        acc += w[((int64_t)co * Cin + ci) * K + j] * x[(int64_t)ci * L + i];
                }
            }
            y[(int64_t)co * Lout + l] = acc;
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * D3  ConvTranspose1d = the exact adjoint of D2 (BASELINE.json configs[0]: "a mirrored
 * ConvTranspose1d stack"):
 *     y[co][m] = b[co] + sum_ci sum_{(l,j): s*l + j - p = m} w[ci][co][j] * x[ci][l],
 *     m in [0, L_out),  L_out = (L-1)*s - 2p + K + op.
 * Written as the scatter it is defined by: every input sample adds its K weighted copies.
 * x: [Cin][L], w: [Cin][Cout][K], y: [Cout][L_out].
 * -------------------------------------------------------------------------------------------*/
int gwo_convt1d_lout(int L, int K, int s, int p, int op) { return (L - 1) * s - 2 * p + K + op; }

void gwo_conv_transpose1d(const double *x, const double *w, const double *b, int Cin, int Cout,
                          int L, int K, int s, int p, int op, double *y) {
    int Lout = gwo_convt1d_lout(L, K, s, p, op);
#pragma omp parallel for schedule(static)
    for (int co = 0; co < Cout; ++co) {
        double *yc = y + (int64_t)co * Lout;
        for (int m = 0; m < Lout; ++m) yc[m] = b ? b[co] : 0.0;
        for (int ci = 0; ci < Cin; ++ci) {
            for (int l = 0; l < L; ++l) {
                for (int j = 0; j < K; ++j) {
                    int m = s * l + j - p;
                    if (m >= 0 && m < Lout)
                        yc[m] += w[((int64_t)ci * Cout + co) * K + j] * x[(int64_t)ci * L + l];
                }
            }
        }
    }
}

/* ---------------------------------------------------------------------------------------------
 * D4  BatchNorm, inference form (BASELINE.json configs[1]: "folded BatchNorm"; reading A6):
 *     z -> gamma*(z - mean)/sqrt(var + eps) + beta   per channel, between conv and activation.
 * gwo_batchnorm applies it unfolded; gwo_bn_fold_* produce the folded weights
 *     w' = w*g,  b' = (b - mean)*g + beta,  g = gamma/sqrt(var + eps)
 * (g indexes dim 0 of a Conv1d weight [Cout][Cin][K], dim 1 of a ConvTranspose1d weight
 * [Cin][Cout][K]).  The two are pinned against each other to 1e-12.
 * -------------------------------------------------------------------------------------------*/
void gwo_batchnorm(double *z, int C, int L, const double *gamma, const double *beta,
                   const double *mean, const double *var, double eps) {
    for (int c = 0; c < C; ++c)
        for (int l = 0; l < L; ++l)
            z[(int64_t)c * L + l] =
                gamma[c] * (z[(int64_t)c * L + l] - mean[c]) / sqrt(var[c] + eps) + beta[c];
}

void gwo_bn_fold_conv(double *w, double *b, int Cout, int Cin, int K, const double *gamma,
                      const double *beta, const double *mean, const double *var, double eps) {
    for (int co = 0; co < Cout; ++co) {
        double g = gamma[co] / sqrt(var[co] + eps);
        for (int ci = 0; ci < Cin; ++ci)
            for (int j = 0; j < K; ++j) w[((int64_t)co * Cin + ci) * K + j] *= g;
        b[co] = (b[co] - mean[co]) * g + beta[co];
    }
}

void gwo_bn_fold_convt(double *w, double *b, int Cin, int Cout, int K, const double *gamma,
                       const double *beta, const double *mean, const double *var, double eps) {
    for (int co = 0; co < Cout; ++co) {
        double g = gamma[co] / sqrt(var[co] + eps);
        for (int ci = 0; ci < Cin; ++ci)
            for (int j = 0; j < K; ++j) w[((int64_t)ci * Cout + co) * K + j] *= g;
        b[co] = (b[co] - mean[co]) * g + beta[co];
    }
}

/* ---------------------------------------------------------------------------------------------
 * D5  Activations (BASELINE.json: tanh in DeepClean, ReLU + sigmoid in the classifier), libm.
 * act: 0 none, 1 tanh, 2 ReLU.
 * -------------------------------------------------------------------------------------------*/
void gwo_activation(double *z, int64_t n, int act) {
    for (int64_t i = 0; i < n; ++i) {
        if (act == 1) z[i] = tanh(z[i]);
        else if (act == 2) z[i] = z[i] > 0.0 ? z[i] : 0.0;
    }
}

double gwo_sigmoid(double z) { return 1.0 / (1.0 + exp(-z)); }

/* ---------------------------------------------------------------------------------------------
 * D6  MaxPool1d(pool, stride = pool), global average pooling, dense layer (BASELINE.json
 * configs[2]: "maxpool 4, then global average pooling, dense 128->64->1 and a sigmoid").
 * -------------------------------------------------------------------------------------------*/
void gwo_maxpool1d(const double *x, int C, int L, int pool, double *y) {
    int Lq = L / pool;
    for (int c = 0; c < C; ++c)
        for (int q = 0; q < Lq; ++q) {
            double m = x[(int64_t)c * L + (int64_t)pool * q];
            for (int i = 1; i < pool; ++i) {
                double v = x[(int64_t)c * L + (int64_t)pool * q + i];
                if (v > m) m = v;
            }
            y[(int64_t)c * Lq + q] = m;
        }
}

void gwo_gap(const double *x, int C, int L, double *y) {
    for (int c = 0; c < C; ++c) {
        double s = 0.0;
        for (int l = 0; l < L; ++l) s += x[(int64_t)c * L + l];
        y[c] = s / (double)L;
    }
}

void gwo_dense(const double *x, const double *w, const double *b, int Cin, int Cout, double *y) {
    for (int co = 0; co < Cout; ++co) {
        double s = b ? b[co] : 0.0;
        for (int ci = 0; ci < Cin; ++ci) s += w[(int64_t)co * Cin + ci] * x[ci];
        y[co] = s;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Storage-type rounding (reading A9/A18: "bf16 weights", BASELINE.json configs[1]; the quantised
 * weights ARE the model, so the oracle takes weights rounded to the storage type and widened
 * back to double).  Round-to-nearest, ties-to-even, straight from double to the target grid:
 * p = significand bits incl. the hidden one (bf16 8, fp16 11, fp32 24), emin = min normal exponent.
 * dtype: 0 bf16, 1 fp16, 2 fp32.  Values beyond the largest finite number become +-inf.
 * Relies on the default rounding mode (nearest-even) of nearbyint().
 * -------------------------------------------------------------------------------------------*/
double gwo_round_scalar(double v, int dtype) {
    int p = dtype == 0 ? 8 : (dtype == 1 ? 11 : 24);
    int emin = dtype == 1 ? -14 : -126;
    int emax = dtype == 1 ? 15 : 127;
    if (v == 0.0 || isnan(v) || isinf(v)) return v;
    int e;
    frexp(v, &e);          /* |v| = f * 2^e, f in [0.5, 1)  ->  floor(log2|v|) = e - 1 */
    e -= 1;
    if (e < emin) e = emin; /* subnormal range: fixed spacing 2^(emin-p+1) */
    double ulp = ldexp(1.0, e - (p - 1));
    double r = nearbyint(v / ulp) * ulp;
    double maxv = (2.0 - ldexp(1.0, -(p - 1))) * ldexp(1.0, emax);
    if (fabs(r) > maxv) return v > 0 ? INFINITY : -INFINITY;
    return r;
}

void gwo_round_storage(double *a, int64_t n, int dtype) {
    for (int64_t i = 0; i < n; ++i) a[i] = gwo_round_scalar(a[i], dtype);
}

/* ---------------------------------------------------------------------------------------------
 * D7  Hann overlap-add (BASELINE.json north_star (3) "overlap-add, window normalisation and
 * subtraction"; motivated by PAPER.md:166/:180 "potential for improved performance by
 * aggregating overlapping predictions").  Periodic Hann (reading A10):
 *     w[n] = 1/2 - 1/2 cos(2 pi n / W).
 * Window t covers absolute samples a = (t+1)S - W + n.  Accumulators over absolute index a >= 0:
 *     acc[a] += w[n] * p_t[n],   wsum[a] += w[n]          (samples a < 0 are never output)
 * Running estimate nhat_t[a] = acc_t[a]/wsum_t[a];  cleaned_t[a] = strain[a] - nhat_t[a]
 * ("subtracts", "postprocessed then subtracted from the associated
 * strain data").
 * -------------------------------------------------------------------------------------------*/
void gwo_hann(int W, double *w) {
    for (int n = 0; n < W; ++n) w[n] = 0.5 - 0.5 * cos(2.0 * M_PI * (double)n / (double)W);
}

/* add window t's weighted prediction into acc/wsum (arrays over absolute index [0, T)) */
void gwo_ola_accumulate(double *acc, double *wsum, int64_t T, const double *p, const double *w,
                        int64_t first_index, int W) {
    for (int n = 0; n < W; ++n) {
        int64_t a = first_index + n;
        if (a < 0 || a >= T) continue;
        acc[a] += w[n] * p[n];
        wsum[a] += w[n];
    }
}

/* cleaned[a] = strain[a] - acc[a]/wsum[a] for a in [a0, a1); positions a < 0 give 0 (A12) and
 * positions never covered by a window (wsum == 0) pass the strain through. */
void gwo_cleaned(const double *acc, const double *wsum, const float *strain, int64_t a0,
                 int64_t a1, double *nhat, double *cleaned) {
    for (int64_t a = a0; a < a1; ++a) {
        int64_t i = a - a0;
        if (a < 0) { nhat[i] = 0.0; cleaned[i] = 0.0; continue; }
        double nh = wsum[a] > 0.0 ? acc[a] / wsum[a] : 0.0;
        nhat[i] = nh;
        cleaned[i] = (double)strain[a] - nh;
    }
}
