"""Shapes of the five BASELINE.json configurations (C0..C4) as plain data.

No arithmetic of the method lives here: only layer shapes, window/stride sizes and
channel-role maps.  The paper itself gives no layer shapes ("a 1-D
convolutional autoencoder", "1-D convolutional neural networks"); they come
from BASELINE.json configs[0..2], with the readings A3-A6, A15 of DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

ACT_NONE, ACT_TANH, ACT_RELU = 0, 1, 2
KIND_CONV, KIND_CONVT = 0, 1
DT_BF16, DT_FP16 = 0, 1
AGG_HANN_OLA, AGG_LAST_STRIDE = 0, 1


@dataclass(frozen=True)
class ConvSpec:
    kind: int          # KIND_CONV (Conv1d) or KIND_CONVT (ConvTranspose1d)
    cin: int
    cout: int
    k: int
    stride: int
    pad_l: int         # Conv1d: left zero padding; ConvTranspose1d: `padding`
    pad_r: int         # Conv1d: right zero padding; ConvTranspose1d: `output_padding`
    act: int
    bn: bool = False   # BatchNorm between conv and activation (folded at load time)
    pool: int = 1      # MaxPool1d(pool, stride=pool) after the activation (classifier only)

    def lout(self, lin: int) -> int:
        if self.kind == KIND_CONV:
            return ((lin + self.pad_l + self.pad_r - self.k) // self.stride + 1) // self.pool
        return (lin - 1) * self.stride - 2 * self.pad_l + self.k + self.pad_r

    def fan_in(self) -> float:
        if self.kind == KIND_CONV:
            return float(self.cin * self.k)
        return self.cin * self.k / self.stride   # taps that reach one output (reading A7)

    def wshape(self) -> Tuple[int, int, int]:
        if self.kind == KIND_CONV:
            return (self.cout, self.cin, self.k)
        return (self.cin, self.cout, self.k)


def deepclean_layers(widths: List[int], bn: bool, k: int = 7) -> List[ConvSpec]:
    """Encoder Conv1d widths[0]->...->widths[-1] (k, stride 2, pad k//2, tanh) and the mirrored
    ConvTranspose1d decoder ending in 1 channel with a linear output (readings A3-A6)."""
    p = k // 2
    layers = []
    for cin, cout in zip(widths[:-1], widths[1:]):
        layers.append(ConvSpec(KIND_CONV, cin, cout, k, 2, p, p, ACT_TANH, bn))
    dec = list(reversed(widths))
    dec[-1] = 1
    for i, (cin, cout) in enumerate(zip(dec[:-1], dec[1:])):
        last = i == len(dec) - 2
        layers.append(ConvSpec(KIND_CONVT, cin, cout, k, 2, p, 1,
                               ACT_NONE if last else ACT_TANH, bn and not last))
    return layers


def bbh_layers(widths=(2, 32, 64, 128), k: int = 8, pool: int = 4) -> List[ConvSpec]:
    """Classifier conv blocks: Conv1d stride 1, 'same' padding pL=3,pR=4, ReLU, MaxPool1d(4) (A15)."""
    pl = (k - 1) // 2
    pr = k - 1 - pl
    return [ConvSpec(KIND_CONV, cin, cout, k, 1, pl, pr, ACT_RELU, False, pool)
            for cin, cout in zip(widths[:-1], widths[1:])]


@dataclass(frozen=True)
class StreamSpec:
    n_streams: int
    n_det: int            # detectors per stream
    fs: int
    window: int           # W, samples
    stride: int           # S, samples
    n_witness: int = 21

    @property
    def channels(self) -> int:          # rows of the snapshot ring per stream (A17)
        return self.n_det * (self.n_witness + 1)

    def witness_rows(self, det: int) -> List[int]:
        base = det * (self.n_witness + 1)
        return list(range(base, base + self.n_witness))

    def strain_row(self, det: int) -> int:
        return det * (self.n_witness + 1) + self.n_witness


@dataclass(frozen=True)
class Config:
    name: str
    stream: StreamSpec
    dc_layers: List[ConvSpec]
    bbh_convs: List[ConvSpec] = field(default_factory=list)
    bbh_dense: Tuple[int, ...] = ()      # (128, 64, 1)
    bbh_len: int = 0                     # classifier window L_b in samples (D8)
    n_updates: int = 0
    seed: int = 0


def config_c0() -> Config:
    return Config("C0", StreamSpec(1, 1, 512, 512, 64), deepclean_layers([21, 8, 16, 32], bn=False),
                  n_updates=32, seed=0)


def config_c1(stride: int = 1024) -> Config:
    return Config("C1", StreamSpec(1, 1, 4096, 32768, stride),
                  deepclean_layers([21, 32, 64, 128, 256], bn=True), n_updates=40, seed=1)


def config_c2() -> Config:
    return Config("C2", StreamSpec(1, 2, 4096, 4096, 4096), [], bbh_layers(), (128, 64, 1), 4096,
                  n_updates=0, seed=2)


def config_c3(n_streams: int = 1, stride: int = 512, window: int = 32768) -> Config:
    return Config("C3" if n_streams == 1 else "C4", StreamSpec(n_streams, 2, 4096, window, stride),
                  deepclean_layers([21, 32, 64, 128, 256], bn=True), bbh_layers(), (128, 64, 1), 4096,
                  n_updates=4800, seed=3)


def config_small_ensemble(n_streams: int = 2) -> Config:
    """A scaled-down C3 (same structure, every stage present) that the oracle runs in seconds:
    W=2048, S=256 (k=8), classifier window 1024.  Used by tests and smoke()."""
    return Config("C3-small", StreamSpec(n_streams, 2, 4096, 2048, 256),
                  deepclean_layers([21, 32, 64, 128, 256], bn=True), bbh_layers(), (128, 64, 1), 1024,
                  n_updates=12, seed=5)
