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
    o = binding.Options(conv_impl=5, fuse_tail=0, pdl=0, snake=0, two_sm=0, skip_zeros=0, incremental=1, fuse_bbh=0)
    L.gw_options_default(C.byref(o))
    assert (o.conv_impl, o.fuse_tail, o.pdl, o.snake, o.two_sm, o.skip_zeros, o.incremental, o.fuse_bbh) == (0, 1, 1, 1, 1, 1, 0, 1)
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
