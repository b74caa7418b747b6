"""Thin ctypes binding over libgwstream.so (include/gwstream.h).  Argument marshalling only:
every step of the path runs in the library's CUDA kernels.  torch is used for device memory and
streams.  There is no fallback: if the library (or a CUDA device) is missing, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

from . import specs as S

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgwstream.so")

GW_OK, GW_EINVAL, GW_ESTATE, GW_ENOMEM, GW_ECUDA = 0, -1, -2, -3, -4
GW_BF16, GW_FP16 = 0, 1
GW_FINAL, GW_RUNNING = 0, 1
GW_IMPL_UMMA, GW_IMPL_SIMT = 0, 1

EXPORTS = [          # include/gwstream.h
    "gw_last_error", "gw_kernel_launches", "gw_options_default",
    "gw_stream_create", "gw_stream_destroy", "gw_stream_update", "gw_stream_snapshot", "gw_stream_count",
    "gw_deepclean_create", "gw_deepclean_destroy", "gw_deepclean_forward", "gw_deepclean_noise",
    "gw_cleaned_strain", "gw_noise_estimate", "gw_deepclean_activation",
    "gw_bbh_create", "gw_bbh_destroy", "gw_bbh_score", "gw_bbh_score_batch",
    "gw_pipeline_create", "gw_pipeline_destroy", "gw_step", "gw_step_host", "gw_step_host_async", "gw_pipeline_graph_nodes",
    "gw_deepclean_set_scaling", "gw_offline_set_scaling", "gw_deepclean_set_postfilter", "gw_bbh_set_whitening", "gw_offline_create", "gw_offline_destroy", "gw_offline_samples", "gw_offline_run", "gw_offline_predictions",
    "gw_ola_offline_noalloc",
]
DIAG_EXPORTS = [     # include/gwstream_diag.h (measurement and diagnostics, not the product interface)
    "gw_step_profile", "gw_profile_label", "gw_profile_flops", "gw_profile_smem_bytes", "gw_probe_mma_cycles", "gw_probe_mufu_rate",
    "gw_incremental_zones", "gw_bbh_fused_images",
]

_FP = C.POINTER(C.c_float)


class Options(C.Structure):
    """gw_options (include/gwstream.h): everything that selects a code path, fixed when a handle is created.
    Defaults: tensor-core kernels, fused tail, PDL, snake order, CTA pairs, zero skipping on; incremental off; the
    classifier as one shared-memory-resident kernel (fuse_bbh) on."""
    _fields_ = [("conv_impl", C.c_int), ("fuse_tail", C.c_int), ("pdl", C.c_int), ("snake", C.c_int),
                ("two_sm", C.c_int), ("skip_zeros", C.c_int), ("incremental", C.c_int), ("fuse_bbh", C.c_int), ("fuse_head", C.c_int)]

    def __init__(self, **kw):
        super().__init__()
        self.conv_impl, self.fuse_tail, self.pdl, self.snake, self.two_sm, self.skip_zeros, self.incremental = \
            GW_IMPL_UMMA, 1, 1, 1, 1, 1, 0
        self.fuse_bbh = 1
        self.fuse_head = 1
        for k, v in kw.items():
            if k not in dict(self._fields_):
                raise TypeError(f"unknown option {k}")
            setattr(self, k, int(v))


def _opt_ptr(opts):
    return None if opts is None else C.byref(opts)


class _ConvLayer(C.Structure):
    _fields_ = [("kind", C.c_int), ("cin", C.c_int), ("cout", C.c_int), ("k", C.c_int), ("stride", C.c_int),
                ("pad_l", C.c_int), ("pad_r", C.c_int), ("act", C.c_int), ("pool", C.c_int),
                ("w", _FP), ("b", _FP), ("bn_gamma", _FP), ("bn_beta", _FP), ("bn_mean", _FP), ("bn_var", _FP),
                ("bn_eps", C.c_float)]


class _DcSpec(C.Structure):
    _fields_ = [("n_det", C.c_int), ("n_layers", C.c_int), ("n_witness", C.c_int),
                ("layers", C.POINTER(_ConvLayer)), ("witness_rows", C.POINTER(C.c_int)),
                ("strain_row", C.POINTER(C.c_int)), ("agg", C.c_int), ("delta", C.c_int)]


class _BbhSpec(C.Structure):
    _fields_ = [("n_convs", C.c_int), ("convs", C.POINTER(_ConvLayer)), ("n_dense", C.c_int),
                ("dense_dims", C.POINTER(C.c_int)), ("dense_w", C.POINTER(_FP)), ("dense_b", C.POINTER(_FP)),
                ("length", C.c_int)]


class GwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gwstream error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libgwstream.so; raises (loudly) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2108_12430_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, i64 = C.c_void_p, C.c_int, C.c_int64
        L.gw_last_error.restype = C.c_char_p
        L.gw_last_error.argtypes = [vp]
        L.gw_kernel_launches.restype = i64
        L.gw_options_default.argtypes = [C.POINTER(Options)]
        L.gw_options_default.restype = None
        L.gw_probe_mma_cycles.argtypes = [i, C.POINTER(C.c_float), C.POINTER(C.c_float)]
        L.gw_probe_mufu_rate.argtypes = [i, i, C.POINTER(C.c_float)]
        L.gw_incremental_zones.argtypes = [C.POINTER(_ConvLayer), i, i, C.POINTER(i), C.POINTER(i)]
        L.gw_bbh_fused_images.argtypes = [C.POINTER(_BbhSpec), i, vp, vp, vp]
        L.gw_stream_create.argtypes = [C.POINTER(vp), i, i, i, i, i]
        L.gw_stream_destroy.argtypes = [vp]
        L.gw_stream_update.argtypes = [vp, vp, vp]
        L.gw_stream_snapshot.argtypes = [vp, vp, C.POINTER(i64), vp]
        L.gw_stream_count.argtypes = [vp]
        L.gw_stream_count.restype = i64
        L.gw_deepclean_create.argtypes = [C.POINTER(vp), vp, C.POINTER(_DcSpec), i, C.POINTER(Options)]
        L.gw_deepclean_destroy.argtypes = [vp]
        L.gw_deepclean_forward.argtypes = [vp, vp]
        L.gw_deepclean_noise.argtypes = [vp, vp, vp]
        L.gw_cleaned_strain.argtypes = [vp, vp, i, vp]
        L.gw_noise_estimate.argtypes = [vp, vp, vp]
        L.gw_deepclean_activation.argtypes = [vp, i, vp, i64, C.POINTER(i), C.POINTER(i), vp]
        L.gw_bbh_create.argtypes = [C.POINTER(vp), vp, C.POINTER(_BbhSpec), i, i, i, C.POINTER(Options)]
        L.gw_bbh_destroy.argtypes = [vp]
        L.gw_bbh_score.argtypes = [vp, vp, vp]
        L.gw_bbh_score_batch.argtypes = [vp, vp, i, vp, vp]
        L.gw_pipeline_create.argtypes = [C.POINTER(vp), vp, vp, vp]
        L.gw_pipeline_destroy.argtypes = [vp]
        L.gw_step.argtypes = [vp, vp, vp, vp, vp]
        L.gw_step_host.argtypes = [vp, vp, vp, vp, vp]
        L.gw_step_host_async.argtypes = [vp, vp, vp, vp, vp]
        L.gw_deepclean_set_scaling.argtypes = [vp, vp, vp, vp, vp]
        L.gw_offline_set_scaling.argtypes = [vp, vp, vp, vp, vp]
        L.gw_deepclean_set_postfilter.argtypes = [vp, vp, i]
        L.gw_bbh_set_whitening.argtypes = [vp, vp, i]
        L.gw_offline_create.argtypes = [C.POINTER(vp), vp, i, i, i, i, i, i, C.POINTER(Options)]
        L.gw_offline_destroy.argtypes = [vp]
        L.gw_offline_samples.argtypes = [vp]
        L.gw_offline_samples.restype = i64
        L.gw_offline_run.argtypes = [vp, vp, vp, vp, vp]
        L.gw_offline_predictions.argtypes = [vp, vp, vp]
        L.gw_ola_offline_noalloc.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, vp]
        L.gw_pipeline_graph_nodes.argtypes = [vp]
        L.gw_step_profile.argtypes = [vp, vp, vp, vp, vp, i, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                      C.POINTER(C.c_double), C.POINTER(i)]
        L.gw_profile_label.argtypes = [vp, i]
        L.gw_profile_label.restype = C.c_char_p
        L.gw_profile_flops.argtypes = [vp, i]
        L.gw_profile_flops.restype = C.c_double
        L.gw_profile_smem_bytes.argtypes = [vp, i]
        L.gw_profile_smem_bytes.restype = C.c_double
        _lib = L
    return _lib


def _check(rc: int, handle=None) -> None:
    if rc != GW_OK:
        raise GwError(rc, lib().gw_last_error(handle).decode())


def kernel_launches() -> int:
    return int(lib().gw_kernel_launches())


def bbh_fused_images(convs: Sequence[S.ConvSpec], conv_params, dense_dims: Sequence[int], length: int, dtype: int):
    """Host only: the operand images (uint16 arrays w1 [128][64], w2 [4][64][64], w3 [8][128][64], still swizzled) of the
    one-kernel classifier as gw_bbh_create builds them (gwstream_diag.h)."""
    keep: list = []
    arr = _marshal_layers(convs, conv_params, keep)
    dims_c = (C.c_int * len(dense_dims))(*dense_dims)
    spec = _BbhSpec(len(convs), arr, len(dense_dims) - 1, dims_c, None, None, length)
    w1 = np.zeros((128, 64), np.uint16); w2 = np.zeros((4, 64, 64), np.uint16); w3 = np.zeros((8, 128, 64), np.uint16)
    _check(lib().gw_bbh_fused_images(C.byref(spec), dtype, C.c_void_p(w1.ctypes.data), C.c_void_p(w2.ctypes.data),
                                     C.c_void_p(w3.ctypes.data)))
    return w1, w2, w3


def incremental_zones(layer_specs: Sequence[S.ConvSpec], stride: int):
    """(left, right) output-position counts per layer that an incremental update recomputes (gwstream_diag.h)."""
    arr = (_ConvLayer * len(layer_specs))()
    for a, l in zip(arr, layer_specs):
        a.kind, a.cin, a.cout, a.k, a.stride, a.pad_l, a.pad_r, a.act, a.pool = \
            l.kind, l.cin, l.cout, l.k, l.stride, l.pad_l, l.pad_r, l.act, l.pool
    n = len(layer_specs)
    left, right = (C.c_int * n)(), (C.c_int * n)()
    _check(lib().gw_incremental_zones(arr, n, int(stride), left, right))
    return list(left), list(right)


def probe_mma_cycles(n_values=(16, 32, 64, 128, 256)):
    """Diagnostic: {N: (issue cycles, completion cycles) per tcgen05.mma} measured on the current device.

        python -c "from paper_2108_12430_b200 import binding as gw; gw.print_mma_probe()"
    """
    out = {}
    for n in n_values:
        a, b = C.c_float(0), C.c_float(0)
        _check(lib().gw_probe_mma_cycles(int(n), C.byref(a), C.byref(b)))
        out[int(n)] = (float(a.value), float(b.value))
    return out


def probe_mufu_rate(mode: int = 0, threads: int = 512) -> float:
    """Diagnostic: activation results per clock per SM (gwstream_diag.h; mode 0 tanh.f32, 1 tanh.f16x2, 2 ex2 + rcp)."""
    r = C.c_float(0)
    _check(lib().gw_probe_mufu_rate(int(mode), int(threads), C.byref(r)))
    return float(r.value)


def print_mma_probe() -> None:
    for n, (issue, done) in probe_mma_cycles().items():
        print(f"N={n:3d}: issue {issue:6.1f} clk/MMA, complete {done:6.1f} clk/MMA  (math floor {n // 2}, shared-memory "
              f"operand read 32 + N/4 = {32 + n // 4})")


def _fp(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(_FP)


def _stream_ptr(stream) -> C.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _ptr(t) -> C.c_void_p:
    return C.c_void_p(0 if t is None else t.data_ptr())


def _marshal_layers(layer_specs: Sequence[S.ConvSpec], params: Sequence[Dict[str, np.ndarray]], keep: list):
    arr = (_ConvLayer * len(layer_specs))()
    for i, (l, p) in enumerate(zip(layer_specs, params)):
        w = np.ascontiguousarray(p["w"], dtype=np.float32)
        b = np.ascontiguousarray(p["b"], dtype=np.float32)
        assert w.shape == l.wshape(), (w.shape, l.wshape())
        keep += [w, b]
        a = arr[i]
        a.kind, a.cin, a.cout, a.k, a.stride = l.kind, l.cin, l.cout, l.k, l.stride
        a.pad_l, a.pad_r, a.act, a.pool = l.pad_l, l.pad_r, l.act, l.pool
        a.w, a.b = _fp(w), _fp(b)
        if l.bn:
            bn = [np.ascontiguousarray(p[k], dtype=np.float32) for k in ("bn_gamma", "bn_beta", "bn_mean", "bn_var")]
            keep += bn
            a.bn_gamma, a.bn_beta, a.bn_mean, a.bn_var = (_fp(x) for x in bn)
            a.bn_eps = float(p["bn_eps"])
    return arr


class Stream:
    """Snapshotter state for n independent streams."""

    def __init__(self, spec: S.StreamSpec):
        self.spec = spec
        self.h = C.c_void_p()
        _check(lib().gw_stream_create(C.byref(self.h), spec.n_streams, spec.channels, spec.fs, spec.window, spec.stride))

    def update(self, new_samples, stream=None) -> None:
        """new_samples: CUDA float32 tensor [n][C][S], contiguous."""
        sp = self.spec
        assert new_samples.is_cuda and new_samples.is_contiguous() and new_samples.dtype.is_floating_point
        assert tuple(new_samples.shape) == (sp.n_streams, sp.channels, sp.stride), tuple(new_samples.shape)
        _check(lib().gw_stream_update(self.h, _ptr(new_samples), _stream_ptr(stream)), self.h)

    def snapshot(self, stream=None):
        import torch
        sp = self.spec
        out = torch.empty((sp.n_streams, sp.channels, sp.window), dtype=torch.float32, device="cuda")
        first = C.c_int64(0)
        _check(lib().gw_stream_snapshot(self.h, _ptr(out), C.byref(first), _stream_ptr(stream)), self.h)
        return out, int(first.value)

    def count(self) -> int:
        return int(lib().gw_stream_count(self.h))

    def close(self) -> None:
        if self.h:
            lib().gw_stream_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _scaling_args(*arrays):
    keep = [None if a is None else np.ascontiguousarray(a, dtype=np.float32) for a in arrays]
    ptrs = [C.c_void_p(0) if a is None else C.c_void_p(a.ctypes.data) for a in keep]
    ptrs[0]._keep = keep                                  # the arrays outlive the call
    return ptrs


class DeepClean:
    """One DeepClean network per detector over a Stream."""

    def __init__(self, stream: Stream, layers: Sequence[S.ConvSpec], params_per_det: Sequence[Sequence[Dict]],
                 dtype: int = GW_BF16, agg: int = S.AGG_HANN_OLA, delta: int = 0, opts: Optional[Options] = None):
        sp = stream.spec
        self.stream, self.layers, self.dtype = stream, list(layers), dtype
        keep: list = []
        n_det = len(params_per_det)
        assert n_det == sp.n_det
        flat_specs = list(layers) * n_det
        flat_params = [p for det in params_per_det for p in det]
        arr = _marshal_layers(flat_specs, flat_params, keep)
        wit = (C.c_int * (n_det * sp.n_witness))(*[r for d in range(n_det) for r in sp.witness_rows(d)])
        srow = (C.c_int * n_det)(*[sp.strain_row(d) for d in range(n_det)])
        spec = _DcSpec(n_det, len(layers), sp.n_witness, arr, wit, srow, agg, delta)
        self.h = C.c_void_p()
        _check(lib().gw_deepclean_create(C.byref(self.h), stream.h, C.byref(spec), dtype, _opt_ptr(opts)), stream.h)

    def set_scaling(self, wit_mean=None, wit_std=None, strain_mean=None, strain_std=None) -> None:
        """Per-channel standardisation of the witnesses ([D][n_witness]) and rescaling of the estimate ([D]);
        None = identity.  Before the first update."""
        _check(lib().gw_deepclean_set_scaling(self.h, *_scaling_args(wit_mean, wit_std, strain_mean, strain_std)), self.h)

    def set_postfilter(self, taps) -> None:
        """D11: causal FIR over the stream of emitted (final) estimate samples; None switches it off.  Before the first update."""
        if taps is None:
            _check(lib().gw_deepclean_set_postfilter(self.h, None, 0), self.h)
            return
        t = np.ascontiguousarray(taps, dtype=np.float32).reshape(-1)
        _check(lib().gw_deepclean_set_postfilter(self.h, C.c_void_p(t.ctypes.data), len(t)), self.h)

    def forward(self, stream=None) -> None:
        _check(lib().gw_deepclean_forward(self.h, _stream_ptr(stream)), self.h)

    def noise(self, stream=None):
        import torch
        sp = self.stream.spec
        out = torch.empty((sp.n_streams, sp.n_det, sp.window), dtype=torch.float32, device="cuda")
        _check(lib().gw_deepclean_noise(self.h, _ptr(out), _stream_ptr(stream)), self.h)
        return out

    def cleaned(self, mode: int = GW_FINAL, stream=None):
        import torch
        sp = self.stream.spec
        n = sp.stride if mode == GW_FINAL else sp.window
        out = torch.empty((sp.n_streams, sp.n_det, n), dtype=torch.float32, device="cuda")
        _check(lib().gw_cleaned_strain(self.h, _ptr(out), mode, _stream_ptr(stream)), self.h)
        return out

    def noise_estimate(self, stream=None):
        import torch
        sp = self.stream.spec
        out = torch.empty((sp.n_streams, sp.n_det, sp.window), dtype=torch.float32, device="cuda")
        _check(lib().gw_noise_estimate(self.h, _ptr(out), _stream_ptr(stream)), self.h)
        return out

    def activation(self, layer: int, stream=None):
        """Stored activations after `layer` (-1 = the gathered window): [n][D][L][C_padded], 16-bit."""
        import torch
        sp = self.stream.spec
        rows, cols = C.c_int(0), C.c_int(0)
        _check(lib().gw_deepclean_activation(self.h, layer, None, 0, C.byref(rows), C.byref(cols), _stream_ptr(stream)), self.h)
        tdt = torch.bfloat16 if self.dtype == GW_BF16 else torch.float16
        out = torch.empty((sp.n_streams, sp.n_det, rows.value, cols.value), dtype=tdt, device="cuda")
        _check(lib().gw_deepclean_activation(self.h, layer, _ptr(out), out.numel() * 2, None, None, _stream_ptr(stream)), self.h)
        return out

    def close(self) -> None:
        if self.h:
            lib().gw_deepclean_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Bbh:
    """BBH classifier, attached to a DeepClean stage or stateless."""

    def __init__(self, dc: Optional[DeepClean], convs: Sequence[S.ConvSpec], conv_params, dense_params,
                 length: int, dtype: int = GW_BF16, n_det: int = 2, max_batch: int = 256, opts: Optional[Options] = None):
        keep: list = []
        arr = _marshal_layers(convs, conv_params, keep)
        dims = [dense_params[0]["w"].shape[1]] + [p["w"].shape[0] for p in dense_params]
        dims_c = (C.c_int * len(dims))(*dims)
        ws = [np.ascontiguousarray(p["w"], dtype=np.float32) for p in dense_params]
        bs = [np.ascontiguousarray(p["b"], dtype=np.float32) for p in dense_params]
        keep += ws + bs
        w_c = (_FP * len(ws))(*[_fp(w) for w in ws])
        b_c = (_FP * len(bs))(*[_fp(b) for b in bs])
        spec = _BbhSpec(len(convs), arr, len(dense_params), dims_c, w_c, b_c, length)
        self.dc, self.length, self.n_det, self.max_batch = dc, length, n_det, max_batch
        self.h = C.c_void_p()
        _check(lib().gw_bbh_create(C.byref(self.h), dc.h if dc is not None else None, C.byref(spec), dtype,
                                   n_det, max_batch, _opt_ptr(opts)))

    def set_whitening(self, taps) -> None:
        """D12: causal FIR whitening of each detector's classifier window, taps [n_det][n_taps]; None switches it off."""
        if taps is None:
            _check(lib().gw_bbh_set_whitening(self.h, None, 0), self.h)
            return
        t = np.ascontiguousarray(taps, dtype=np.float32)
        assert t.ndim == 2 and t.shape[0] == self.n_det, t.shape
        _check(lib().gw_bbh_set_whitening(self.h, C.c_void_p(t.ctypes.data), t.shape[1]), self.h)

    def score(self, stream=None):
        import torch
        out = torch.empty((self.dc.stream.spec.n_streams,), dtype=torch.float32, device="cuda")
        _check(lib().gw_bbh_score(self.h, _ptr(out), _stream_ptr(stream)), self.h)
        return out

    def score_batch(self, windows, stream=None):
        import torch
        assert windows.is_cuda and windows.is_contiguous() and windows.dtype == torch.float32
        B = windows.shape[0]
        assert tuple(windows.shape[1:]) == (self.n_det, self.length)
        out = torch.empty((B,), dtype=torch.float32, device="cuda")
        _check(lib().gw_bbh_score_batch(self.h, _ptr(windows), B, _ptr(out), _stream_ptr(stream)), self.h)
        return out

    def close(self) -> None:
        if self.h:
            lib().gw_bbh_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Pipeline:
    """update -> forward -> cleaned -> score as one CUDA-graph replay per stride."""

    def __init__(self, stream: Stream, dc: DeepClean, bbh: Optional[Bbh]):
        self.stream, self.dc, self.bbh = stream, dc, bbh
        self.h = C.c_void_p()
        _check(lib().gw_pipeline_create(C.byref(self.h), stream.h, dc.h, bbh.h if bbh is not None else None))

    def step(self, new_samples, scores, cleaned_final, stream=None) -> None:
        """All CUDA float32 tensors: new [n][C][S], scores [n], cleaned_final [n][D][S]."""
        _check(lib().gw_step(self.h, _ptr(new_samples), _ptr(scores), _ptr(cleaned_final), _stream_ptr(stream)), self.h)

    def step_host(self, new_samples, scores, cleaned_final, stream=None) -> None:
        """Host tensors / numpy float32 arrays (pinned for asynchronous copies)."""
        def hp(a):
            if a is None:
                return C.c_void_p(0)
            return C.c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())
        _check(lib().gw_step_host(self.h, hp(new_samples), hp(scores), hp(cleaned_final), _stream_ptr(stream)), self.h)

    def step_host_async(self, new_samples, scores, cleaned_final, stream=None) -> None:
        """step_host without the synchronisation: the input copy of this call overlaps the previous step's
        kernels.  All three host buffers must stay untouched until `stream` is synchronised past the call."""
        def hp(a):
            if a is None:
                return C.c_void_p(0)
            return C.c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())
        _check(lib().gw_step_host_async(self.h, hp(new_samples), hp(scores), hp(cleaned_final), _stream_ptr(stream)), self.h)

    def step_profile(self, new_samples, scores, cleaned_final, stream=None):
        """One update through the profiling graph (gwstream_diag.h): the kernels gw_step replays, each stamping
        %globaltimer at its first CTA's start and last CTA's end.  -> [dict(label, begin_us, end_us, flops, smem_bytes)]
        in launch order; begin/end are relative to the start of the step's first kernel."""
        n_max = 32
        b, e, mhz = (C.c_double * n_max)(), (C.c_double * n_max)(), (C.c_double * n_max)()
        n = C.c_int(0)
        _check(lib().gw_step_profile(self.h, _ptr(new_samples), _ptr(scores), _ptr(cleaned_final),
                                     _stream_ptr(stream), n_max, b, e, mhz, C.byref(n)), self.h)
        return [{"label": lib().gw_profile_label(self.h, i).decode(), "begin_us": float(b[i]), "end_us": float(e[i]),
                 "sm_mhz": float(mhz[i]),
                 "flops": float(lib().gw_profile_flops(self.h, i)), "smem_bytes": float(lib().gw_profile_smem_bytes(self.h, i))}
                for i in range(min(n.value, n_max))]

    def graph_nodes(self) -> int:
        return int(lib().gw_pipeline_graph_nodes(self.h))

    def close(self) -> None:
        if self.h:
            lib().gw_pipeline_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Offline:
    """Offline / non-streaming DeepClean (D9): `n_windows` consecutive windows of ONE stream's archival
    segment per launch.  `spec` gives the per-stream shape (n_streams is ignored)."""

    def __init__(self, spec: S.StreamSpec, layers: Sequence[S.ConvSpec], params_per_det: Sequence[Sequence[Dict]],
                 n_windows: int, dtype: int = GW_BF16, opts: Optional[Options] = None):
        self.spec, self.n_windows = spec, n_windows
        keep: list = []
        n_det = len(params_per_det)
        assert n_det == spec.n_det
        arr = _marshal_layers(list(layers) * n_det, [p for det in params_per_det for p in det], keep)
        wit = (C.c_int * (n_det * spec.n_witness))(*[r for d in range(n_det) for r in spec.witness_rows(d)])
        srow = (C.c_int * n_det)(*[spec.strain_row(d) for d in range(n_det)])
        dspec = _DcSpec(n_det, len(layers), spec.n_witness, arr, wit, srow, S.AGG_HANN_OLA, 0)
        self.h = C.c_void_p()
        _check(lib().gw_offline_create(C.byref(self.h), C.byref(dspec), spec.channels, spec.fs, spec.window, spec.stride,
                                       n_windows, dtype, _opt_ptr(opts)))
        self.samples = int(lib().gw_offline_samples(self.h))

    def set_scaling(self, wit_mean=None, wit_std=None, strain_mean=None, strain_std=None) -> None:
        _check(lib().gw_offline_set_scaling(self.h, *_scaling_args(wit_mean, wit_std, strain_mean, strain_std)), self.h)

    def run(self, samples, cleaned=None, noise=None, stream=None):
        """samples: CUDA float32 [C][T]; returns (cleaned [D][T], noise estimate [D][T])."""
        import torch
        assert tuple(samples.shape) == (self.spec.channels, self.samples) and samples.is_contiguous()
        if cleaned is None:
            cleaned = torch.empty((self.spec.n_det, self.samples), dtype=torch.float32, device="cuda")
        if noise is None:
            noise = torch.empty((self.spec.n_det, self.samples), dtype=torch.float32, device="cuda")
        _check(lib().gw_offline_run(self.h, _ptr(samples), _ptr(cleaned), _ptr(noise), _stream_ptr(stream)), self.h)
        return cleaned, noise

    def predictions(self, stream=None):
        import torch
        out = torch.empty((self.n_windows, self.spec.n_det, self.spec.window), dtype=torch.float32, device="cuda")
        _check(lib().gw_offline_predictions(self.h, _ptr(out), _stream_ptr(stream)), self.h)
        return out

    def __del__(self):
        try:
            if self.h:
                lib().gw_offline_destroy(self.h)
                self.h = C.c_void_p()
        except Exception:
            pass


GW_OLA_NOALLOC_MAX_WINDOW = 32768


def ola_offline_noalloc(pred, strain, stride: int, cleaned=None, noise=None, post=None, stream=None):
    """gw_ola_offline_noalloc (include/gwstream.h): the offline Hann overlap-add with the library's built-in scratch,
    no handle and no allocation inside the library.  pred: CUDA float32 [B][D][W]; strain: [D][T], T = W + (B-1)*stride;
    post: optional [D][2] (scale, offset).  Pass `cleaned` (and `noise`) to keep this wrapper from allocating as well.
    Returns (cleaned, noise)."""
    import torch
    B, D, W = (int(v) for v in pred.shape)
    T = W + (B - 1) * int(stride)
    assert pred.is_contiguous() and pred.dtype == torch.float32
    assert tuple(strain.shape) == (D, T) and strain.is_contiguous() and strain.dtype == torch.float32
    if cleaned is None:
        cleaned = torch.empty((D, T), dtype=torch.float32, device=pred.device)
    assert tuple(cleaned.shape) == (D, T) and cleaned.is_contiguous()
    if noise is not None:
        assert tuple(noise.shape) == (D, T) and noise.is_contiguous()
    if post is not None:
        assert tuple(post.shape) == (D, 2) and post.is_contiguous() and post.dtype == torch.float32
    _check(lib().gw_ola_offline_noalloc(_ptr(pred), _ptr(strain), _ptr(cleaned), _ptr(noise), _ptr(post), B, D, W, int(stride),
                                        _stream_ptr(stream)))
    return cleaned, noise


def build_ensemble(cfg: S.Config, dc_params_per_det, bbh_params=None, dtype: int = GW_BF16,
                   agg: int = S.AGG_HANN_OLA, delta: int = 0, opts: Optional[Options] = None):
    """Convenience: Stream + DeepClean (+ Bbh) + Pipeline for a specs.Config."""
    st = Stream(cfg.stream)
    dc = DeepClean(st, cfg.dc_layers, dc_params_per_det, dtype, agg, delta, opts)
    bbh = None
    if bbh_params is not None:
        cp, dp = bbh_params
        bbh = Bbh(dc, cfg.bbh_convs, cp, dp, cfg.bbh_len, dtype, opts=opts)
    pipe = Pipeline(st, dc, bbh)
    return st, dc, bbh, pipe
