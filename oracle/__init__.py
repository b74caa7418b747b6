"""CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Double-precision, definition-by-definition statement of the hot path of arXiv:2108.12430
(see gw_oracle.c for the per-function citations and DESIGN.md for the definitions D1..D8 and
the readings A1..A23).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline and
--impl reference legs may import this package.  It never imports paper_2108_12430_b200.

Layer descriptions are duck-typed: any object with attributes
``kind (0 Conv1d | 1 ConvTranspose1d), cin, cout, k, stride, pad_l, pad_r, act (0 none | 1 tanh |
2 ReLU), bn, pool`` (for ConvTranspose1d pad_l = padding, pad_r = output_padding).

Parity pins: tests/test_oracle_pins.py (none of the functions here is "parity unpinned").
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gw_oracle.c")
_LIB = os.path.join(_HERE, "libgw_oracle.so")

KIND_CONV, KIND_CONVT = 0, 1
ACT_NONE, ACT_TANH, ACT_RELU = 0, 1, 2
DT_BF16, DT_FP16, DT_FP32 = 0, 1, 2
AGG_HANN_OLA, AGG_LAST_STRIDE = 0, 1


def build(force: bool = False) -> str:
    """Compile gw_oracle.c with gcc -O2 (+OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-std=c11", "-D_GNU_SOURCE",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None
_D = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_F = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        i, i64, dbl, vp = C.c_int, C.c_int64, C.c_double, C.c_void_p
        L.gwo_num_threads.restype = i
        L.gwo_set_num_threads.argtypes = [i]
        L.gwo_snapshot.argtypes = [_F, i, i64, i64, i, i, _F, C.POINTER(i64)]
        L.gwo_conv1d_lout.argtypes = [i] * 5
        L.gwo_conv1d_lout.restype = i
        L.gwo_convt1d_lout.argtypes = [i] * 5
        L.gwo_convt1d_lout.restype = i
        L.gwo_conv1d.argtypes = [_D, _D, vp, i, i, i, i, i, i, i, _D]
        L.gwo_conv_transpose1d.argtypes = [_D, _D, vp, i, i, i, i, i, i, i, _D]
        L.gwo_batchnorm.argtypes = [_D, i, i, _D, _D, _D, _D, dbl]
        L.gwo_bn_fold_conv.argtypes = [_D, _D, i, i, i, _D, _D, _D, _D, dbl]
        L.gwo_bn_fold_convt.argtypes = [_D, _D, i, i, i, _D, _D, _D, _D, dbl]
        L.gwo_activation.argtypes = [_D, i64, i]
        L.gwo_sigmoid.argtypes = [dbl]
        L.gwo_sigmoid.restype = dbl
        L.gwo_maxpool1d.argtypes = [_D, i, i, i, _D]
        L.gwo_gap.argtypes = [_D, i, i, _D]
        L.gwo_dense.argtypes = [_D, _D, vp, i, i, _D]
        L.gwo_round_scalar.argtypes = [dbl, i]
        L.gwo_round_scalar.restype = dbl
        L.gwo_round_storage.argtypes = [_D, i64, i]
        L.gwo_hann.argtypes = [i, _D]
        L.gwo_ola_accumulate.argtypes = [_D, _D, i64, _D, _D, i64, i]
        L.gwo_cleaned.argtypes = [_D, _D, _F, i64, i64, _D, _D]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().gwo_num_threads())


def set_num_threads(n: int) -> None:
    lib().gwo_set_num_threads(int(n))


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _bptr(b: Optional[np.ndarray]):
    return None if b is None else b.ctypes.data_as(C.c_void_p)


# ---------------------------------------------------------------------------------- primitives

def snapshot(x_all: np.ndarray, t: int, S: int, W: int):
    """D1.  x_all [C][T] float32 with T >= (t+1)S.  -> ([C][W] float32, first index)."""
    x_all = np.ascontiguousarray(x_all, dtype=np.float32)
    Cn, T = x_all.shape
    assert T >= (t + 1) * S
    out = np.empty((Cn, W), dtype=np.float32)
    first = C.c_int64(0)
    lib().gwo_snapshot(x_all, Cn, T, t, S, W, out, C.byref(first))
    return out, int(first.value)


def conv1d(x, w, b=None, stride=1, pad_l=0, pad_r=0) -> np.ndarray:
    """D2.  x [Cin][L], w [Cout][Cin][K] -> [Cout][Lout] float64."""
    x, w = _d(x), _d(w)
    b = None if b is None else _d(b)
    Cout, Cin, K = w.shape
    assert x.shape[0] == Cin
    L = x.shape[1]
    Lout = lib().gwo_conv1d_lout(L, K, stride, pad_l, pad_r)
    y = np.empty((Cout, Lout), dtype=np.float64)
    lib().gwo_conv1d(x, w, _bptr(b), Cin, Cout, L, K, stride, pad_l, pad_r, y)
    return y


def conv_transpose1d(x, w, b=None, stride=1, pad=0, out_pad=0) -> np.ndarray:
    """D3.  x [Cin][L], w [Cin][Cout][K] -> [Cout][Lout] float64."""
    x, w = _d(x), _d(w)
    b = None if b is None else _d(b)
    Cin, Cout, K = w.shape
    assert x.shape[0] == Cin
    L = x.shape[1]
    Lout = lib().gwo_convt1d_lout(L, K, stride, pad, out_pad)
    y = np.empty((Cout, Lout), dtype=np.float64)
    lib().gwo_conv_transpose1d(x, w, _bptr(b), Cin, Cout, L, K, stride, pad, out_pad, y)
    return y


def batchnorm(z, gamma, beta, mean, var, eps) -> np.ndarray:
    """D4, unfolded."""
    z = _d(z).copy()
    lib().gwo_batchnorm(z, z.shape[0], z.shape[1], _d(gamma), _d(beta), _d(mean), _d(var), float(eps))
    return z


def bn_fold(kind: int, w, b, gamma, beta, mean, var, eps):
    """D4, folded form.  Returns (w', b') float64."""
    w, b = _d(w).copy(), _d(b).copy()
    if kind == KIND_CONV:
        Cout, Cin, K = w.shape
        lib().gwo_bn_fold_conv(w, b, Cout, Cin, K, _d(gamma), _d(beta), _d(mean), _d(var), float(eps))
    else:
        Cin, Cout, K = w.shape
        lib().gwo_bn_fold_convt(w, b, Cin, Cout, K, _d(gamma), _d(beta), _d(mean), _d(var), float(eps))
    return w, b


def activation(z, act: int) -> np.ndarray:
    z = _d(z).copy()
    lib().gwo_activation(z.reshape(-1), z.size, act)
    return z


def sigmoid(z: float) -> float:
    return float(lib().gwo_sigmoid(float(z)))


def maxpool1d(x, pool: int) -> np.ndarray:
    x = _d(x)
    y = np.empty((x.shape[0], x.shape[1] // pool), dtype=np.float64)
    lib().gwo_maxpool1d(x, x.shape[0], x.shape[1], pool, y)
    return y


def gap(x) -> np.ndarray:
    x = _d(x)
    y = np.empty((x.shape[0],), dtype=np.float64)
    lib().gwo_gap(x, x.shape[0], x.shape[1], y)
    return y


def dense(x, w, b=None) -> np.ndarray:
    x, w = _d(x), _d(w)
    b = None if b is None else _d(b)
    y = np.empty((w.shape[0],), dtype=np.float64)
    lib().gwo_dense(x, w, _bptr(b), w.shape[1], w.shape[0], y)
    return y


def round_storage(a, dtype: int) -> np.ndarray:
    """RN-even to the bf16 / fp16 / fp32 grid, result widened to float64 (A9, A18)."""
    a = _d(a).copy()
    lib().gwo_round_storage(a.reshape(-1), a.size, dtype)
    return a


def hann(W: int) -> np.ndarray:
    """Periodic Hann w[n] = 1/2 - 1/2 cos(2 pi n / W) (D7, A10)."""
    w = np.empty((W,), dtype=np.float64)
    lib().gwo_hann(W, w)
    return w


def fir_causal(x, taps) -> np.ndarray:
    """D11 / D12: causal FIR with zero initial state along the last axis, y[i] = sum_{j < len(taps)} taps[j] x[i - j],
    x[i < 0] = 0.  Written out as the definition (one shifted, scaled copy of x per tap), float64.
    (DESIGN.md readings: PAPER.md:198 "the noise frame is postprocessed then subtracted", :212 "cleaned strains are
    combined and postprocessed then passed to BBHnet"; the paper defines neither operation.)"""
    x = _d(x)
    taps = _d(taps).reshape(-1)
    y = np.zeros_like(x)
    n = x.shape[-1]
    for j in range(len(taps)):
        if j >= n:
            break
        y[..., j:] += taps[j] * x[..., :n - j]
    return y


# ------------------------------------------------------------------------------------- models

def prepare_conv(layer, params: Dict[str, np.ndarray], dtype: int):
    """Storage-precision folded parameters of one conv layer (A9): BatchNorm folded in float64
    (D4), weights rounded RN-even to `dtype`, bias rounded to fp32, both widened to float64."""
    w, b = _d(params["w"]), _d(params["b"])
    if getattr(layer, "bn", False):
        w, b = bn_fold(layer.kind, w, b, params["bn_gamma"], params["bn_beta"], params["bn_mean"],
                       params["bn_var"], float(params["bn_eps"]))
    return round_storage(w, dtype), round_storage(b, DT_FP32)


def prepare_dense(params: Dict[str, np.ndarray]):
    """Dense head parameters are stored in fp32."""
    return round_storage(params["w"], DT_FP32), round_storage(params["b"], DT_FP32)


def conv_layer(x, layer, w, b) -> np.ndarray:
    """One layer: conv (D2/D3) -> activation (D5) -> max-pool (D6), BatchNorm already folded."""
    if layer.kind == KIND_CONV:
        y = conv1d(x, w, b, layer.stride, layer.pad_l, layer.pad_r)
    else:
        y = conv_transpose1d(x, w, b, layer.stride, layer.pad_l, layer.pad_r)
    y = activation(y, layer.act)
    if getattr(layer, "pool", 1) > 1:
        y = maxpool1d(y, layer.pool)
    return y


def deepclean_forward(x, layers: Sequence, prepared: Sequence, return_all: bool = False,
                      act_dtype: Optional[int] = None):
    """x [n_witness][W] -> predicted noise p [W] (DeepClean takes the witness
    channels and predicts the noise in the strain).  prepared[i] = prepare_conv(layers[i], ...).

    act_dtype (DIAGNOSTIC ONLY, not the oracle of record): when given, the input and every
    inter-layer activation are rounded RN-even to that storage type, i.e. the result an exact
    machine would get if it had to store activations in 16 bits.  It separates the storage
    rounding that any 16-bit implementation must incur from implementation error (DESIGN.md,
    "Error budget")."""
    h = _d(x)
    if act_dtype is not None:
        h = round_storage(h, act_dtype)
    acts = []
    for i, (layer, (w, b)) in enumerate(zip(layers, prepared)):
        h = conv_layer(h, layer, w, b)
        if act_dtype is not None and i < len(layers) - 1:
            h = round_storage(h, act_dtype)
        if return_all:
            acts.append(h)
    assert h.shape[0] == 1
    return (h[0], acts) if return_all else h[0]


def bbh_forward(x, convs: Sequence, prepared_convs: Sequence, prepared_dense: Sequence,
                return_logit: bool = False):
    """x [2][L_b] -> score in (0,1) (BBHnet on the cleaned strain of both
    detectors gives an event likelihood).  conv blocks -> GAP -> dense+ReLU ... -> dense -> sigmoid."""
    h = _d(x)
    for layer, (w, b) in zip(convs, prepared_convs):
        h = conv_layer(h, layer, w, b)
    v = gap(h)
    for i, (w, b) in enumerate(prepared_dense):
        v = dense(v, w, b)
        if i < len(prepared_dense) - 1:
            v = activation(v, ACT_RELU)
    assert v.shape == (1,)
    return float(v[0]) if return_logit else sigmoid(float(v[0]))


# ----------------------------------------------------------------------------------- streaming

class StreamOracle:
    """One stream of the end-to-end ensemble, update by update, in the paper's order
    (PAPER.md:76 Fig. 4, :212): snapshotter -> one DeepClean per detector -> aggregation and
    subtraction -> classifier on the cleaned strain of all detectors.

    rows: per detector, (list of witness row indices, strain row index) into the [C] channel axis.
    dc: per detector, (layers, prepared).  bbh: None or (convs, prepared_convs, prepared_dense, L_b).
    agg: AGG_HANN_OLA (D7, default, north_star (3)) or AGG_LAST_STRIDE (the paper's causal scheme,
    PAPER.md:182: "predicted segments keep only their most recent floor(fs/r) samples").
    delta: aggregation-latency offset in samples, used by D8 and AGG_LAST_STRIDE.
    """

    def __init__(self, channels: int, W: int, S: int, rows, dc, bbh=None, agg: int = AGG_HANN_OLA,
                 delta: int = 0, max_updates: int = 64, scaling=None, postfilter=None, whiten=None):
        # postfilter (D11): None or FIR taps [Lh] applied, causally and with carried state, to the
        # STREAM of emitted (final) estimate samples before rescaling and subtraction; running values are not filtered.
        # whiten (D12): None or FIR taps [D][Lg] applied to each detector's classifier window with zero
        # initial state at the window start.
        self.postfilter = None if postfilter is None else _d(postfilter).reshape(-1)
        self.whiten = None if whiten is None else _d(whiten)
        # scaling (reading A14): None or (wit_mean [D][n_wit], wit_std [D][n_wit],
        # strain_mean [D], strain_std [D]): the network sees (x - mean) / std of every witness and the
        # aggregated estimate is subtracted as strain_std * nhat + strain_mean.
        self.scaling = scaling
        self.C, self.W, self.S = channels, W, S
        self.rows, self.dc, self.bbh, self.agg, self.delta = rows, dc, bbh, agg, delta
        self.T = max_updates * S
        self.x = np.zeros((channels, self.T), dtype=np.float32)   # every sample so far
        self.t = -1
        ndet = len(rows)
        self.acc = np.zeros((ndet, self.T), dtype=np.float64)
        self.wsum = np.zeros((ndet, self.T), dtype=np.float64)
        self.emitted = np.zeros((ndet, self.T), dtype=np.float64)   # D11: emitted estimate samples over absolute index
        self.w = hann(W)

    def _cleaned(self, d: int, strain_all: np.ndarray, a0: int, a1: int):
        """Estimate and cleaned strain of samples [a0, a1) of detector d (zeros before the stream start);
        post-processing (A14): where an estimate exists it is rescaled to strain_std * nhat + strain_mean."""
        nh = np.empty(a1 - a0); cl = np.empty(a1 - a0)
        lib().gwo_cleaned(self.acc[d], self.wsum[d], strain_all, a0, a1, nh, cl)
        if self.scaling is not None:
            a = np.arange(a0, a1)
            ok = (a >= 0) & (a < self.T)
            has = np.zeros(a1 - a0, dtype=bool)
            has[ok] = self.wsum[d][a[ok]] > 0
            nh = np.where(has, float(self.scaling[3][d]) * nh + float(self.scaling[2][d]), nh)
            cl = np.where(has, strain_all[np.clip(a, 0, self.T - 1)].astype(np.float64) - nh, cl)
        return nh, cl

    def _final_postfiltered(self, d: int, strain_all: np.ndarray, fin0: int, S: int):
        """D11: this update's emitted block joins the stream of emitted estimate samples (unscaled, zeros before the
        stream start); the stream is FIR-filtered causally (carried state = the earlier emitted samples), then rescaled
        (A14) and subtracted.  Samples with negative absolute index give 0 (A12)."""
        saved, self.scaling = self.scaling, None
        raw, _ = self._cleaned(d, strain_all, fin0, fin0 + S)              # unscaled estimate of the emitted block
        self.scaling = saved
        nh = np.zeros(S); cl = np.zeros(S)
        for i in range(S):
            a = fin0 + i
            if a < 0:
                continue
            self.emitted[d][a] = raw[i]
        for i in range(S):
            a = fin0 + i
            if a < 0:
                continue
            acc = 0.0
            for j, hj in enumerate(self.postfilter):
                if a - j >= 0:
                    acc += hj * self.emitted[d][a - j]
            if self.scaling is not None:
                acc = float(self.scaling[3][d]) * acc + float(self.scaling[2][d])
            nh[i] = acc
            cl[i] = float(strain_all[a]) - acc
        return nh, cl

    def skip(self, new: np.ndarray) -> None:
        """Append an update's samples WITHOUT computing it (tests that check a late block of a long stream: the
        windows of later updates then hold the true history, while the overlap-add state lacks the skipped windows --
        final values are valid again once W/S computed updates have passed, D7)."""
        self.t += 1
        assert (self.t + 1) * self.S <= self.T, "raise max_updates"
        self.x[:, self.t * self.S:(self.t + 1) * self.S] = new

    def update(self, new: np.ndarray) -> Dict[str, np.ndarray]:
        """new [C][S] float32, strictly new samples.  Returns this update's results."""
        W, S = self.W, self.S
        self.t += 1
        t = self.t
        assert (t + 1) * S <= self.T, "raise max_updates"
        self.x[:, t * S:(t + 1) * S] = new
        snap, first = snapshot(self.x[:, :(t + 1) * S], t, S, W)              # D1
        out = {"snapshot": snap, "first_index": first, "pred": [], "nhat_final": [], "cleaned_final": [],
               "nhat_running": [], "cleaned_running": []}
        count = (t + 1) * S
        for d, ((wit, srow), (layers, prepared)) in enumerate(zip(self.rows, self.dc)):
            xin_d = snap[wit].astype(np.float64)
            if self.scaling is not None:                                            # pre-processing (A14)
                xin_d = (xin_d - _d(self.scaling[0])[d][:, None]) / _d(self.scaling[1])[d][:, None]
                xin_d[:, :max(0, -first)] = 0.0      # before the stream start the network sees zeros (A12), not -mean/std
            p = deepclean_forward(xin_d, layers, prepared)                          # D2-D5
            out["pred"].append(p)
            strain_all = np.ascontiguousarray(self.x[srow])
            if self.agg == AGG_HANN_OLA:                                            # D7
                lib().gwo_ola_accumulate(self.acc[d], self.wsum[d], self.T, _d(p), self.w, first, W)
                acc, wsum = self.acc[d], self.wsum[d]
                fin0 = first                      # the S samples that became final this update
            else:
                a0 = count - S - self.delta
                for n in range(W - S - self.delta, W - self.delta):
                    a = first + n
                    if 0 <= a < self.T:
                        self.acc[d][a] = p[n]
                        self.wsum[d][a] = 1.0
                acc, wsum = self.acc[d], self.wsum[d]
                fin0 = a0
            nh, cl = self._cleaned(d, strain_all, fin0, fin0 + S)
            if self.postfilter is not None:                                         # D11
                nh, cl = self._final_postfiltered(d, strain_all, fin0, S)
            out["nhat_final"].append(nh); out["cleaned_final"].append(cl)
            nhr, clr = self._cleaned(d, strain_all, first, first + W)
            out["nhat_running"].append(nhr); out["cleaned_running"].append(clr)
        if self.bbh is not None:                                                    # D8
            convs, pc, pd, Lb = self.bbh
            a1 = count - self.delta
            xin = np.zeros((len(self.rows), Lb), dtype=np.float64)
            for d, (wit, srow) in enumerate(self.rows):
                _, xin[d] = self._cleaned(d, np.ascontiguousarray(self.x[srow]), a1 - Lb, a1)
            if self.whiten is not None:                                             # D12
                xin = np.stack([fir_causal(xin[d], self.whiten[d]) for d in range(len(self.rows))])
            out["bbh_input"] = xin
            out["score"] = bbh_forward(xin, convs, pc, pd)
        return out


def offline_clean(x: np.ndarray, W: int, S: int, rows, dc, scaling=None) -> Dict[str, np.ndarray]:
    """D9, offline / non-streaming mode ("adjacent frames ... in parallel",
    :202 offline regime, :216 non-streaming ensemble): an archival segment x [C][T], T = W + (B-1) S, of ONE
    stream is cut into the B windows [jS, jS + W) that lie inside it -- the same window grid as the streaming
    path (D1), without the warm-up windows that reach before the segment -- every window goes through DeepClean
    independently, and the predictions are combined by the same periodic-Hann overlap-add (D7), normalised by
    the summed weights of the windows that actually cover a sample:

        nhat[a] = sum_j w[a - jS] p_j[a - jS] / sum_j w[a - jS]   (j: jS <= a < jS + W, 0 <= j < B)
        cleaned[d][a] = strain_d[a] - nhat_d[a]

    A sample covered by all W/S windows gets exactly the streaming path's final value.  Sample 0 is covered
    only at window position 0, where the periodic Hann weight is 0: its estimate is defined as 0.
    Returns {"pred": [D][B][W], "nhat": [D][T], "cleaned": [D][T]} in float64."""
    x = np.asarray(x)
    C, T = x.shape
    assert T >= W and (T - W) % S == 0
    B = (T - W) // S + 1
    w = hann(W)
    ndet = len(rows)
    pred = np.zeros((ndet, B, W), dtype=np.float64)
    nhat = np.zeros((ndet, T), dtype=np.float64)
    cleaned = np.zeros((ndet, T), dtype=np.float64)
    for d, ((wit, strain), (layers, prepared)) in enumerate(zip(rows, dc)):
        acc = np.zeros(T, dtype=np.float64)
        wsum = np.zeros(T, dtype=np.float64)
        for j in range(B):
            xin = x[wit, j * S:j * S + W].astype(np.float64)
            if scaling is not None:                       # pre-processing (A14), as in StreamOracle
                xin = (xin - _d(scaling[0])[d][:, None]) / _d(scaling[1])[d][:, None]
            p = deepclean_forward(xin, layers, prepared)
            pred[d, j] = p
            acc[j * S:j * S + W] += w * p
            wsum[j * S:j * S + W] += w
        ok = wsum > 0
        nhat[d, ok] = acc[ok] / wsum[ok]
        if scaling is not None:                           # post-processing where an estimate exists
            nhat[d, ok] = float(scaling[3][d]) * nhat[d, ok] + float(scaling[2][d])
        cleaned[d] = x[strain].astype(np.float64) - nhat[d]
    return {"pred": pred, "nhat": nhat, "cleaned": cleaned}
