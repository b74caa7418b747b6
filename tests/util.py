"""Shared helpers for the parity tests: build the oracle and the CUDA engine for the SAME seeded
inputs and raw parameters (paper_2108_12430_b200.synth), and the tolerances of north_star."""
from __future__ import annotations

import numpy as np

import oracle
from paper_2108_12430_b200 import specs as S
from paper_2108_12430_b200 import synth

# north_star tolerances (BASELINE.json): network outputs relative L2 <= 1e-2 and every element
# |d| <= 2e-2 * RMS(oracle output); classifier scores |d| <= 5e-3; snapshots bit-exact.
REL_L2 = 1e-2
ELEM_RMS = 2e-2
SCORE_ABS = 5e-3
# Pure-bf16 activations cannot meet the per-element bar on the 8-layer network, whatever the
# implementation: rounding the activations of the fp64 oracle itself to bf16 at each layer boundary
# already gives max |d| = 2.9e-2..3.8e-2 RMS (tests/test_oracle_pins.py::
# test_bf16_activation_storage_alone_exceeds_the_elementwise_bar).  The
# relative-L2 bar (1e-2) holds for bf16 and is asserted; the per-element bar for bf16 is set to
# 6e-2 RMS = 1.5x the storage-rounding floor, and the CUDA path is additionally held to the
# storage-rounded oracle (see check_against_rounded).  fp16 (the paper's precision)
# is held to north_star's bars as stated.
ELEM_RMS_BF16 = 6e-2


def elem_tol(dtype: int) -> float:
    return ELEM_RMS_BF16 if dtype == 0 else ELEM_RMS


def oracle_dtype(dtype: int) -> int:
    return oracle.DT_BF16 if dtype == 0 else oracle.DT_FP16


LOGIT_ABS = 2e-2      # |d score| <= 5e-3 at the steepest point of the sigmoid <=> |d logit| <= 2e-2


def centred_bbh_params(seed: int, convs, dense, length: int, dtype: int = 0):
    """Random classifier weights put every score near sigmoid(-4), where the 5e-3 score bar would
    accept almost anything.  Shift the last dense bias (a parameter, i.e. an input handed to both
    sides) so that the oracle's mean logit over a few noise windows is 0: scores then spread around
    0.5, where the bar bites."""
    cp, dp = synth.bbh_params(seed, convs, dense)
    od = oracle_dtype(dtype)
    pc = [oracle.prepare_conv(l, p, od) for l, p in zip(convs, cp)]
    pd = [oracle.prepare_dense(p) for p in dp]
    x = synth.bbh_windows(seed + 1, 4, length)
    mean_logit = float(np.mean([oracle.bbh_forward(x[i], convs, pc, pd, return_logit=True) for i in range(4)]))
    dp[-1]["b"] = (dp[-1]["b"] - np.float32(mean_logit)).astype(np.float32)
    return cp, dp


def logit(p):
    p = np.asarray(p, dtype=np.float64)
    return np.log(p / (1.0 - p))


def make_params(cfg: S.Config):
    st = cfg.stream
    dc = [synth.deepclean_params(cfg.seed * 100 + d, cfg.dc_layers) for d in range(st.n_det)] if cfg.dc_layers else []
    bbh = centred_bbh_params(cfg.seed * 100 + 50, cfg.bbh_convs, cfg.bbh_dense, cfg.bbh_len) if cfg.bbh_convs else None
    return dc, bbh


def make_stream_oracle(cfg: S.Config, dc_params, bbh_params, dtype: int, max_updates: int,
                       agg: int = oracle.AGG_HANN_OLA, delta: int = 0, scaling=None):
    st = cfg.stream
    od = oracle_dtype(dtype)
    rows = [(st.witness_rows(d), st.strain_row(d)) for d in range(st.n_det)]
    dc = [(cfg.dc_layers, [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.dc_layers, dc_params[d])])
          for d in range(st.n_det)]
    bbh = None
    if bbh_params is not None:
        cp, dp = bbh_params
        bbh = (cfg.bbh_convs, [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.bbh_convs, cp)],
               [oracle.prepare_dense(p) for p in dp], cfg.bbh_len)
    return oracle.StreamOracle(st.channels, st.window, st.stride, rows, dc, bbh, agg=agg, delta=delta,
                               max_updates=max_updates, scaling=scaling)


def unrounded_conv(layer, params):
    """(w, b) of a layer in float64 with BatchNorm folded but WITHOUT rounding to the storage type: the model before
    weight quantisation.  Used only to report the total distance of the CUDA path to that model (context: by reading A9
    the quantised weights are the model)."""
    w, b = np.asarray(params["w"], np.float64), np.asarray(params["b"], np.float64)
    if getattr(layer, "bn", False):
        w, b = oracle.bn_fold(layer.kind, w, b, params["bn_gamma"], params["bn_beta"], params["bn_mean"],
                              params["bn_var"], float(params["bn_eps"]))
    return w, b


def check_network_output(got: np.ndarray, ref: np.ndarray, what: str, rms_ref: np.ndarray | None = None,
                         elem: float = ELEM_RMS, rel_l2: float = REL_L2):
    """relative L2 <= 1e-2 and max |d| <= 2e-2 * RMS(ref) (RMS of `rms_ref` when given; reading A22)."""
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    base = ref if rms_ref is None else np.asarray(rms_ref, dtype=np.float64).ravel()
    rms = float(np.sqrt(np.mean(base * base)))
    assert np.all(np.isfinite(got)), f"{what}: non-finite values"
    if rms == 0.0:
        assert np.array_equal(got, ref), f"{what}: expected exact zeros"
        return 0.0, 0.0
    d = got - ref
    rel = float(np.sqrt(np.sum(d * d)) / max(np.sqrt(np.sum(base * base)), 1e-300))
    worst = float(np.max(np.abs(d)) / rms)
    assert rel <= rel_l2, f"{what}: relative L2 {rel:.3e} > {rel_l2}"
    assert worst <= elem, f"{what}: max |d|/RMS {worst:.3e} > {elem}"
    return rel, worst
