"""gw_ola_offline_noalloc (include/gwstream.h, csrc/gw_noalloc.cu): the offline Hann overlap-add with its tables in the
library's built-in __device__ scratch array, for callers that cannot call cudaMalloc.  Checked against the existing path
(gw_offline_run, whose tables are cudaMalloc'ed and filled from the host) on the SAME predictions, on calls made one after
the other: the array is shared by every call and keeps the last call's tables, so the calls alternate between two
(window, stride) pairs.  The file sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_2108_12430_b200 import binding as gw
from paper_2108_12430_b200 import specs as S
from paper_2108_12430_b200 import synth
from tests import util

pytestmark = pytest.mark.gpu


def _existing_path(cfg, n_windows, dtype, scaling=None):
    """gw_offline_run on a seeded segment: (strain rows [D][T], predictions [B][D][W], cleaned, estimate, post or None)."""
    sp = cfg.stream
    T = sp.window + (n_windows - 1) * sp.stride
    dc_params, _ = util.make_params(cfg)
    x = torch.from_numpy(synth.stream_channels(cfg.seed + 77, sp, T)).cuda()
    off = gw.Offline(sp, cfg.dc_layers, dc_params, n_windows, dtype)
    post = None
    if scaling is not None:
        strain_mean, strain_std = scaling
        off.set_scaling(None, None, strain_mean, strain_std)
        post = torch.from_numpy(np.stack([strain_std, strain_mean], axis=1).astype(np.float32)).cuda().contiguous()
    cleaned, noise = off.run(x)
    pred = off.predictions()
    torch.cuda.synchronize()
    strain = x[[sp.strain_row(d) for d in range(sp.n_det)]].contiguous()
    return strain, pred, cleaned, noise, post


def _compare(got, want, pred, what):
    """Same arithmetic on the same predictions; only the tables differ in where they were computed (device / host double
    cosine), so the bar is far inside the suite's own (2e-2 of the prediction's RMS per element, tests/util.py)."""
    got, want = got.cpu().numpy(), want.cpu().numpy()
    rms = float(np.sqrt(np.mean(pred.cpu().numpy().astype(np.float64) ** 2)))
    worst = float(np.abs(got.astype(np.float64) - want).max()) / rms
    print(f"no-alloc overlap-add vs gw_offline_run, {what}: worst |d|/RMS {worst:.3e}, "
          f"{int((got != want).sum())} of {got.size} samples not bit-identical")
    assert np.isfinite(got).all()
    assert worst <= 1e-5, (what, worst)


def test_no_alloc_overlap_add_matches_the_existing_path_on_calls_in_a_row():
    cfg_a = S.config_small_ensemble(1)                                    # W = 2048, S = 256, two detectors
    sp_b = S.StreamSpec(1, 2, 4096, 4096, 1024)                           # another (window, stride): the tables must be rewritten
    cfg_b = S.Config("noalloc-b", sp_b, cfg_a.dc_layers, seed=9)
    a = _existing_path(cfg_a, 21, gw.GW_FP16)
    b = _existing_path(cfg_b, 6, gw.GW_FP16, scaling=(np.array([0.25, -0.5], np.float32), np.array([1.5, 0.75], np.float32)))
    cs = torch.cuda.Stream()
    outs = []
    # outputs are allocated by the caller, up front, and poisoned; the four calls follow one another on one stream
    bufs = [(torch.full_like(c[2], float("nan")), torch.full_like(c[3], float("nan"))) for c in (a, b, a, a)]
    torch.cuda.synchronize()
    launches = gw.kernel_launches()
    for (strain, pred, _, _, post), (cl, nz), stride in zip((a, b, a, a), bufs, (256, 1024, 256, 256)):
        outs.append(gw.ola_offline_noalloc(pred, strain, stride, cleaned=cl, noise=nz, post=post, stream=cs))
    cs.synchronize()
    assert gw.kernel_launches() - launches == 12                          # two set-up kernels and the overlap-add, per call
    for i, (ref, what) in enumerate(((a, "first call"), (b, "second call, other window/stride, post scaling"),
                                     (a, "third call, back to the first shape"), (a, "fourth call, same shape again"))):
        _compare(outs[i][0], ref[2], ref[1], what + " (cleaned)")
        _compare(outs[i][1], ref[3], ref[1], what + " (estimate)")
    assert torch.equal(outs[2][0], outs[3][0]) and torch.equal(outs[0][0], outs[2][0])   # the same call gives the same numbers
    # the estimate is optional
    only, none = gw.ola_offline_noalloc(a[1], a[0], 256, stream=cs)
    cs.synchronize()
    assert none is None and torch.equal(only, outs[0][0])


def test_no_alloc_entry_point_rejects_what_its_scratch_cannot_hold():
    W = 2 * gw.GW_OLA_NOALLOC_MAX_WINDOW
    pred = torch.zeros((2, 1, W), device="cuda")
    strain = torch.zeros((1, W + W // 2), device="cuda")
    cleaned = torch.full_like(strain, 7.0)
    launches = gw.kernel_launches()
    with pytest.raises(gw.GwError) as e:
        gw.ola_offline_noalloc(pred, strain, W // 2, cleaned=cleaned)
    assert e.value.code == gw.GW_EINVAL and "exceeds" in str(e.value) and str(gw.GW_OLA_NOALLOC_MAX_WINDOW) in str(e.value)
    with pytest.raises(gw.GwError) as e:                                  # window / stride < 2
        gw.ola_offline_noalloc(pred[:, :, :1024].contiguous()[:1], strain[:, :1024].contiguous(), 1024, cleaned=cleaned[:, :1024].contiguous())
    assert e.value.code == gw.GW_EINVAL
    torch.cuda.synchronize()
    assert gw.kernel_launches() == launches and bool((cleaned == 7.0).all())   # nothing was launched
    # the largest window it serves
    W = gw.GW_OLA_NOALLOC_MAX_WINDOW
    g = torch.Generator(device="cuda").manual_seed(5)
    pred = torch.randn((3, 1, W), device="cuda", generator=g)
    strain = torch.randn((1, W + 2 * (W // 4)), device="cuda", generator=g)
    cleaned, noise = gw.ola_offline_noalloc(pred, strain, W // 4, noise=torch.empty_like(strain))
    torch.cuda.synchronize()
    # property that needs no table: where only window 0 covers a sample (a < stride), weight and normaliser cancel
    first = slice(1, W // 4)
    assert torch.allclose(noise[0, first], pred[0, 0, first], rtol=1e-5, atol=1e-6)
    assert torch.equal(cleaned, strain - noise)
