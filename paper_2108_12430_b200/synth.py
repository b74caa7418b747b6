"""Seeded synthetic inputs and raw (unfolded, unquantised) parameters.

This is the ONE module that both the oracle's tests and the CUDA path's tests draw from.
It contains none of the method's arithmetic (no convolution, BatchNorm fold, rounding to the
storage type, window, overlap-add): it only draws random numbers and shapes them like the
paper's workloads.  The recipe is stated in DESIGN.md ("Input recipe"); the workloads it stands
in for are LIGO O2/O3 strain + witness channels, which are not available.

Everything is float32 as handed to both sides (they each widen / quantise on their own).
"""
from __future__ import annotations

import math
from typing import Dict, List

import numpy as np

from . import specs as S

# --------------------------------------------------------------------------------------
# parameters
# --------------------------------------------------------------------------------------

_GAIN = {S.ACT_TANH: 5.0 / 3.0, S.ACT_RELU: math.sqrt(2.0), S.ACT_NONE: 1.0}


def conv_params(rng: np.random.Generator, spec: S.ConvSpec) -> Dict[str, np.ndarray]:
    """Kaiming-uniform weights (reading A7) and, when spec.bn, BatchNorm statistics (A6)."""
    fan_in = spec.fan_in()
    bound = _GAIN[spec.act] * math.sqrt(3.0 / fan_in)
    w = rng.uniform(-bound, bound, size=spec.wshape()).astype(np.float32)
    bb = 1.0 / math.sqrt(fan_in)
    b = rng.uniform(-bb, bb, size=(spec.cout,)).astype(np.float32)
    p = {"w": w, "b": b}
    if spec.bn:
        p["bn_gamma"] = rng.uniform(0.5, 1.5, size=(spec.cout,)).astype(np.float32)
        p["bn_beta"] = rng.uniform(-0.1, 0.1, size=(spec.cout,)).astype(np.float32)
        p["bn_mean"] = (0.1 * rng.standard_normal(spec.cout)).astype(np.float32)
        p["bn_var"] = rng.uniform(0.5, 1.5, size=(spec.cout,)).astype(np.float32)
        p["bn_eps"] = np.float32(1e-5)
    return p


def dense_params(rng: np.random.Generator, cin: int, cout: int, act: int) -> Dict[str, np.ndarray]:
    bound = _GAIN[act] * math.sqrt(3.0 / cin)
    w = rng.uniform(-bound, bound, size=(cout, cin)).astype(np.float32)
    bb = 1.0 / math.sqrt(cin)
    b = rng.uniform(-bb, bb, size=(cout,)).astype(np.float32)
    return {"w": w, "b": b}


def deepclean_params(seed: int, layers: List[S.ConvSpec]) -> List[Dict[str, np.ndarray]]:
    rng = np.random.default_rng(seed)
    return [conv_params(rng, l) for l in layers]


def bbh_params(seed: int, convs: List[S.ConvSpec], dense=(128, 64, 1)):
    rng = np.random.default_rng(seed)
    cp = [conv_params(rng, l) for l in convs]
    dp = []
    for i, (cin, cout) in enumerate(zip(dense[:-1], dense[1:])):
        last = i == len(dense) - 2
        dp.append(dense_params(rng, cin, cout, S.ACT_NONE if last else S.ACT_RELU))
    return cp, dp


# --------------------------------------------------------------------------------------
# time series
# --------------------------------------------------------------------------------------

def white_channels(seed: int, channels: int, n_samples: int) -> np.ndarray:
    """C0: iid N(0,1) float32, [channels][n_samples]."""
    rng = np.random.default_rng(seed)
    return rng.standard_normal((channels, n_samples)).astype(np.float32)


def _coloured(rng: np.random.Generator, n: int, alpha: float = 0.9) -> np.ndarray:
    from scipy.signal import lfilter
    e = rng.standard_normal(n + 256)
    y = lfilter([1.0 - alpha], [1.0, -alpha], e)[256:]
    return y / math.sqrt((1.0 - alpha) / (1.0 + alpha))     # unit variance in steady state


def detector_channels(seed: int, n_samples: int, fs: int = 4096, n_witness: int = 21,
                      t0: int = 0) -> np.ndarray:
    """C1/C3 detector: rows 0..n_witness-1 = witnesses (coloured Gaussian + 60 Hz mains and two
    harmonics), row n_witness = strain (N(0,1) + linear coupling of the witnesses' line parts);
    the 'power mains and harmonics' picture of PAPER.md:36, :188.  float32 [n_witness+1][n_samples]."""
    rng = np.random.default_rng(seed)
    t = (np.arange(n_samples, dtype=np.float64) + t0) / fs
    amp = rng.uniform(0.0, 1.0, size=(n_witness, 3))
    phase = rng.uniform(0.0, 2 * math.pi, size=(n_witness, 3))
    kappa = rng.uniform(-0.5, 0.5, size=(n_witness,))
    out = np.empty((n_witness + 1, n_samples), dtype=np.float32)
    strain = rng.standard_normal(n_samples)
    for c in range(n_witness):
        line = np.zeros(n_samples)
        for h in range(3):
            line += amp[c, h] * np.sin(2 * math.pi * 60.0 * (h + 1) * t + phase[c, h])
        out[c] = (_coloured(rng, n_samples) + line).astype(np.float32)
        strain += kappa[c] * line
    out[n_witness] = strain.astype(np.float32)
    return out


def stream_channels(seed: int, spec: S.StreamSpec, n_samples: int, white: bool = False) -> np.ndarray:
    """All rows of one stream's snapshot ring, [spec.channels][n_samples] float32 (A17: one ring
    holds every data source of the stream; detector d occupies rows d*(n_witness+1)...)."""
    if white:
        return white_channels(seed, spec.channels, n_samples)
    dets = [detector_channels(seed * 7919 + 31 * d + 1, n_samples, spec.fs, spec.n_witness)
            for d in range(spec.n_det)]
    return np.concatenate(dets, axis=0)


def multi_stream(seed: int, spec: S.StreamSpec, n_samples: int, white: bool = False) -> np.ndarray:
    """[n_streams][channels][n_samples] float32; stream i uses seed+i (C4: 'per-stream seeds')."""
    return np.stack([stream_channels(seed + i, spec, n_samples, white) for i in range(spec.n_streams)])


def bbh_windows(seed: int, n_windows: int = 256, length: int = 4096, fs: int = 4096) -> np.ndarray:
    """C2: [n_windows][2][length] float32 whitened-like N(0,1); even-indexed windows carry a
    chirping sine-Gaussian of network SNR U(8,20), second detector shifted by U(-10,10) ms."""
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((n_windows, 2, length))
    t = np.arange(length) / fs
    for i in range(0, n_windows, 2):
        f0 = rng.uniform(50, 300)
        fdot = rng.uniform(0, 400)
        tau = rng.uniform(0.010, 0.050)
        tc = rng.uniform(0.2, 0.8) * length / fs
        phi = rng.uniform(0, 2 * math.pi)
        dt = rng.uniform(-0.010, 0.010)
        snr = rng.uniform(8, 20)
        hs = []
        for shift in (0.0, dt):
            u = t - tc - shift
            hs.append(np.exp(-u * u / (2 * tau * tau)) * np.sin(2 * math.pi * (f0 * u + 0.5 * fdot * u * u) + phi))
        norm = math.sqrt(sum(float(np.sum(h * h)) for h in hs))
        for d in range(2):
            x[i, d] += snr / norm * hs[d]
    return x.astype(np.float32)
