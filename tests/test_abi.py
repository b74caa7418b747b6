"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/gwstream.h declares; without a CUDA device compute entry points fail loudly (no fallback)."""
import ctypes as C
import os
import re

import pytest

from paper_2108_12430_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(header="gwstream.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gw_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    L = C.CDLL(path)
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"{n} declared in gwstream.h but not exported"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and gwstream.h disagree"
    diag = _declared("gwstream_diag.h")
    for n in diag:
        assert hasattr(L, n), f"{n} declared in gwstream_diag.h but not exported"
    assert sorted(binding.DIAG_EXPORTS) == diag, "binding.DIAG_EXPORTS and gwstream_diag.h disagree"
    # the product header carries no process-global switches and no builder diagnostics
    assert not [n for n in names if n.startswith("gw_set_") or "probe" in n or "profile" in n]


def test_options_defaults_and_per_handle_errors():
    L = binding.lib()
    o = binding.Options(conv_impl=5, fuse_tail=0, pdl=0, snake=0, two_sm=0, skip_zeros=0, incremental=1, fuse_bbh=0, fuse_head=0)
    L.gw_options_default(C.byref(o))
    assert (o.conv_impl, o.fuse_tail, o.pdl, o.snake, o.two_sm, o.skip_zeros, o.incremental, o.fuse_bbh, o.fuse_head) == (0, 1, 1, 1, 1, 1, 0, 1, 1)
    # a failing call without a handle is reported for the calling thread: gw_last_error(NULL)
    h = C.c_void_p()
    assert L.gw_stream_create(C.byref(h), 0, 22, 512, 512, 64) == binding.GW_EINVAL
    assert b"gw_stream_create" in L.gw_last_error(None)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    L = binding.lib()
    h = C.c_void_p()
    rc = L.gw_stream_create(C.byref(h), 1, 22, 512, 512, 64)
    assert rc == binding.GW_ECUDA
    assert b"no CPU fallback" in L.gw_last_error(None)


def test_argument_validation_happens_before_touching_the_device():
    L = binding.lib()
    h = C.c_void_p()
    assert L.gw_stream_create(C.byref(h), 0, 22, 512, 512, 64) == binding.GW_EINVAL
    assert L.gw_stream_create(C.byref(h), 1, 22, 512, 64, 512) == binding.GW_EINVAL      # stride > window
    assert L.gw_stream_create(None, 1, 22, 512, 512, 64) == binding.GW_EINVAL
    lay = binding._ConvLayer()
    z = (C.c_int * 1)()
    assert L.gw_incremental_zones(None, 1, 64, z, z) == binding.GW_EINVAL
    lay.kind, lay.k, lay.stride = 0, 7, 3
    assert L.gw_incremental_zones(C.byref(lay), 1, 64, z, z) == binding.GW_EINVAL          # stride-2 layers only
    assert L.gw_stream_update(None, None, None) == binding.GW_EINVAL
    assert L.gw_stream_count(None) == 0


def test_missing_library_raises(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()


def test_fused_classifier_operand_images_hold_every_weight_where_the_kernel_reads_it():
    """Host logic of the one-kernel classifier (no GPU): gw_bbh_fused_images returns the three tensor-core operand images
    gw_bbh_create uploads.  Unswizzled by the rule the header states, every weight must sit -- rounded to the storage type
    exactly as the oracle rounds it -- at the (row, k) the kernel's index arithmetic reads it from, and nothing else may be
    non-zero: block 1 as a Toeplitz matrix over the 11 samples of an im2col row (tap j of output phase q at sample j + q,
    once for the head and once for the tail of a sample), blocks 2 and 3 as [tap][cout][cin]."""
    import numpy as np
    import oracle
    from paper_2108_12430_b200 import specs as S
    from paper_2108_12430_b200 import synth

    def unswizzle(img):                                   # [..., rows, 64] -> the logical K order
        out = np.empty_like(img)
        rows = img.shape[-2]
        for r in range(rows):
            for c in range(8):
                out[..., r, 8 * c:8 * c + 8] = img[..., r, 8 * (c ^ (r & 7)):8 * (c ^ (r & 7)) + 8]
        return out

    def to_float(bits, dtype):
        if dtype == binding.GW_FP16:
            return bits.view(np.float16).astype(np.float64)
        return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)

    for dtype, od in ((binding.GW_FP16, oracle.DT_FP16), (binding.GW_BF16, oracle.DT_BF16)):
        for n_det, widths in ((2, (2, 32, 64, 128)), (1, (1, 24, 48, 128))):
            convs = S.bbh_layers(widths)
            cp, _ = synth.bbh_params(9, convs, (128, 64, 1))
            w1, w2, w3 = binding.bbh_fused_images(convs, cp, (128, 64, 1), 2048, dtype)
            w1, w2, w3 = (to_float(unswizzle(w), dtype) for w in (w1, w2, w3))
            wq = [oracle.round_storage(p["w"], od) for p in cp]              # [cout][cin][8] on the storage grid
            e1 = np.zeros((128, 64))
            for q in range(4):
                for part in range(2):
                    for ci in range(widths[0]):
                        for j in range(8):
                            e1[q * 32:q * 32 + widths[1], (ci * 2 + part) * 16 + j + q] = wq[0][:, ci, j]
            assert np.array_equal(w1, e1)
            e2 = np.zeros((4, 64, 64))
            for j in range(8):
                e2[j // 2, :widths[2], (j % 2) * 32:(j % 2) * 32 + widths[1]] = wq[1][:, :, j]
            assert np.array_equal(w2, e2)
            e3 = np.zeros((8, 128, 64))
            for j in range(8):
                e3[j, :, :widths[2]] = wq[2][:, :, j]
            assert np.array_equal(w3, e3)
    # shapes that kernel does not take are refused, not mangled
    convs = S.bbh_layers((2, 32, 64, 96))
    cp, _ = synth.bbh_params(9, convs, (96, 64, 1))
    with pytest.raises(binding.GwError):
        binding.bbh_fused_images(convs, cp, (96, 64, 1), 2048, binding.GW_FP16)
    convs = S.bbh_layers((2, 32, 64, 128))
    cp, _ = synth.bbh_params(9, convs, (128, 64, 1))
    with pytest.raises(binding.GwError):
        binding.bbh_fused_images(convs, cp, (128, 64, 1), 1000, binding.GW_FP16)   # window not a multiple of 512
