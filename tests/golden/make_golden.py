"""Writes tests/golden/c0_oracle.txt from the CPU oracle ALONE (imports nothing of the CUDA path).

    python tests/golden/make_golden.py

The paper prints no numeric worked example for any stage of this path (every figure of PAPER.md is a missing
image, e.g. PAPER.md:46, :62, :100; layer shapes exist only in BASELINE.json), so there are no paper values to
store.  This fixture freezes a handful of values of the oracle itself on BASELINE.json configs[0] (seed 0, fp16
storage-rounded weights): a later change to the oracle's arithmetic shows up as a diff of this file and has to be
justified against the paper.  Format: one `key update index value` record per line, value
printed with 17 significant digits.
"""
from __future__ import annotations

import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle                                               # noqa: E402
from paper_2108_12430_b200 import specs as S                # noqa: E402  (shapes only)
from paper_2108_12430_b200 import synth                     # noqa: E402  (seeded inputs only)

UPDATES = (0, 7, 8, 31)
INDICES = (0, 1, 63, 64, 255, 511)


def records():
    cfg = S.config_c0()
    sp = cfg.stream
    params = synth.deepclean_params(cfg.seed * 100, cfg.dc_layers)
    prepared = [oracle.prepare_conv(l, p, oracle.DT_FP16) for l, p in zip(cfg.dc_layers, params)]
    rows = [(sp.witness_rows(0), sp.strain_row(0))]
    x = synth.multi_stream(cfg.seed, sp, cfg.n_updates * sp.stride, white=True)[0]
    so = oracle.StreamOracle(sp.channels, sp.window, sp.stride, rows, [(cfg.dc_layers, prepared)], None,
                             max_updates=cfg.n_updates)
    out = []
    for t in range(cfg.n_updates):
        ref = so.update(x[:, t * sp.stride:(t + 1) * sp.stride])
        if t in UPDATES:
            for i in INDICES:
                out.append(("pred", t, i, float(ref["pred"][0][i])))
                out.append(("cleaned_running", t, i, float(ref["cleaned_running"][0][i])))
            for i in (0, 1, sp.stride - 1):
                out.append(("cleaned_final", t, i, float(ref["cleaned_final"][0][i])))
    return out


if __name__ == "__main__":
    with open(os.path.join(HERE, "c0_oracle.txt"), "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ alone; see that file for what this pins\n")
        for key, t, i, v in records():
            f.write(f"{key} {t} {i} {v:.17g}\n")
    print("wrote", os.path.join(HERE, "c0_oracle.txt"))
