"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs.
Bars (north_star): snapshots and indices bit-exact; network outputs relative L2 <= 1e-2 and every
element |d| <= 2e-2 RMS(oracle output); classifier scores |d| <= 5e-3."""
import numpy as np
import pytest
import torch

import oracle
from paper_2108_12430_b200 import binding as gw
from paper_2108_12430_b200 import specs as S
from paper_2108_12430_b200 import synth
from tests import util

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------- a1 snapshot
@pytest.mark.parametrize("n,C,W,S_", [(1, 22, 512, 64), (3, 5, 96, 7), (2, 44, 4096, 512), (2, 3, 10, 10),
                                      (1, 2, 33, 1), (4, 4, 64, 12), (1, 22, 32768, 1024)])
def test_snapshot_bit_exact(n, C, W, S_):
    spec = S.StreamSpec(n, 1, 512, W, S_, n_witness=C - 1)
    st = gw.Stream(spec)
    n_up = min(3 * (W // S_) + 3, 40)
    x = np.random.default_rng(11).standard_normal((n, C, n_up * S_)).astype(np.float32)
    xd = _dev(x)
    for t in range(n_up):
        st.update(xd[:, :, t * S_:(t + 1) * S_].contiguous())
        if t % 3 == 0 or t == n_up - 1:
            snap, first = st.snapshot()
            snap = snap.cpu().numpy()
            for i in range(n):
                ref, first_ref = oracle.snapshot(x[i][:, :(t + 1) * S_], t, S_, W)
                assert first == first_ref
                assert np.array_equal(snap[i].view(np.uint32), ref.view(np.uint32)), (t, i)
    assert st.count() == n_up * S_


# --------------------------------------------------------------------- DeepClean streaming (C0)
def _run_streaming(cfg, dtype, n_up, white, agg=S.AGG_HANN_OLA, delta=0, check_scores=True, impl=gw.GW_IMPL_UMMA,
                   use_graph=False, incremental=False):
    st_spec = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    x = synth.multi_stream(cfg.seed, st_spec, n_up * st_spec.stride, white=white)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, agg, delta,
                                              gw.Options(conv_impl=impl, incremental=incremental))
    oracles = [util.make_stream_oracle(cfg, dc_params, bbh_params, dtype, n_up, agg, delta)
               for _ in range(st_spec.n_streams)]
    xd = _dev(x)
    stats = {"pred": 0.0, "nhat": 0.0, "score": 0.0}
    et = util.elem_tol(dtype)
    cs = torch.cuda.Stream()
    scores_d = torch.zeros(st_spec.n_streams, device="cuda")
    final_d = torch.zeros((st_spec.n_streams, st_spec.n_det, st_spec.stride), device="cuda")
    for t in range(n_up):
        new = xd[:, :, t * st_spec.stride:(t + 1) * st_spec.stride].contiguous()
        if use_graph:
            with torch.cuda.stream(cs):
                cs.wait_stream(torch.cuda.current_stream())      # `new` was produced on torch's current stream
                pipe.step(new, scores_d, final_d, cs)
            cs.synchronize()
            final = final_d.cpu().numpy()
            scores = scores_d.cpu().numpy() if bbh is not None else None
            pred = dc.noise().cpu().numpy()
            running = nhat = None
        else:
            stream.update(new)
            dc.forward()
            pred = dc.noise().cpu().numpy()
            running = dc.cleaned(gw.GW_RUNNING).cpu().numpy()
            nhat = dc.noise_estimate().cpu().numpy()
            scores = bbh.score().cpu().numpy() if bbh is not None else None
            final = None
        snap, first = stream.snapshot()                  # a1 with the DeepClean stage attached (fused a1 + a2 kernel)
        snap = snap.cpu().numpy()
        for i, orc in enumerate(oracles):
            ref = orc.update(x[i][:, t * st_spec.stride:(t + 1) * st_spec.stride])
            assert first == ref["first_index"] and np.array_equal(snap[i], ref["snapshot"]), ("snapshot", t, i)
            for d in range(st_spec.n_det):
                tag = f"update {t} stream {i} det {d}"
                _, w1 = util.check_network_output(pred[i, d], ref["pred"][d], "pred " + tag, elem=et)
                stats["pred"] = max(stats["pred"], w1)
                rms_n = ref["pred"][d]
                if nhat is not None:
                    _, w2 = util.check_network_output(nhat[i, d], ref["nhat_running"][d], "nhat " + tag, rms_ref=rms_n, elem=et)
                    stats["nhat"] = max(stats["nhat"], w2)
                    # reading A22: cleaned is judged against RMS(noise estimate), not against the strain
                    util.check_network_output(running[i, d], ref["cleaned_running"][d], "cleaned " + tag, rms_ref=rms_n, elem=et)
                if final is not None:
                    util.check_network_output(final[i, d], ref["cleaned_final"][d], "final " + tag, rms_ref=rms_n, elem=et)
            if scores is not None and check_scores:
                assert abs(float(scores[i]) - ref["score"]) <= util.SCORE_ABS, (t, i, float(scores[i]), ref["score"])
                assert abs(util.logit(scores[i]) - util.logit(ref["score"])) <= util.LOGIT_ABS, (t, i, float(scores[i]), ref["score"])
                stats["score"] = max(stats["score"], abs(float(scores[i]) - ref["score"]))
    return stats


@pytest.mark.parametrize("dtype", [gw.GW_BF16, gw.GW_FP16])
def test_c0_streaming_deepclean_matches_oracle(dtype):
    """configs[0]: 1 stream, 21 witnesses + strain, W=512, S=64, 32 updates, N(0,1) samples."""
    cfg = S.config_c0()
    stats = _run_streaming(cfg, dtype, cfg.n_updates, white=True)
    print("C0 worst |d|/RMS:", stats)


def test_odd_stride_uses_the_gather_path_and_matches_oracle():
    """S odd: window positions do not pair up with ring slots, so the 16-bit mirror ring is off and the
    window is re-gathered from the fp32 ring every update (strides down to 2-3 samples)."""
    cfg = S.Config("C0-odd", S.StreamSpec(2, 1, 512, 120, 15), S.config_c0().dc_layers, seed=7)
    _run_streaming(cfg, gw.GW_FP16, 20, white=True)


def test_c0_simt_cross_check_matches_oracle():
    cfg = S.config_c0()
    _run_streaming(cfg, gw.GW_BF16, 10, white=True, impl=gw.GW_IMPL_SIMT)


def test_c0_last_stride_mode_and_latency_offset():
    """PAPER.md:182 causal aggregation, PAPER.md:186 aggregation latency delta."""
    cfg = S.config_c0()
    _run_streaming(cfg, gw.GW_BF16, 14, white=True, agg=S.AGG_LAST_STRIDE, delta=0)
    _run_streaming(cfg, gw.GW_BF16, 14, white=True, agg=S.AGG_LAST_STRIDE, delta=96)
    _run_streaming(cfg, gw.GW_BF16, 14, white=True, agg=S.AGG_HANN_OLA, delta=128)


# ------------------------------------------------------------------------ layer-by-layer check
@pytest.mark.parametrize("fuse", [False, True])
@pytest.mark.parametrize("dtype", [gw.GW_FP16, gw.GW_BF16])
def test_c1_shaped_layers_match_oracle_layer_by_layer(dtype, fuse):
    """The full C1 network (21->32->64->128->256 and back, folded BatchNorm) on a 4096-sample window:
    every stored activation against the oracle's, several M tiles and all channel widths.  fuse=True is
    the production path (layers 0 + 1 in one kernel, last tensor-core layer + final ConvTranspose1d in one kernel: the
    activations inside those kernels are not materialised); fuse=False stores and checks those activations as well."""
    cfg = S.Config("C1-short", S.StreamSpec(2, 1, 4096, 4096, 512), S.config_c1().dc_layers, seed=1)
    dc_params, _ = util.make_params(cfg)
    dc_params2 = [dc_params[0]]
    st = gw.Stream(cfg.stream)
    dc = gw.DeepClean(st, cfg.dc_layers, dc_params2, dtype, opts=gw.Options(fuse_tail=fuse, fuse_head=fuse))
    fused_layers = (0, len(cfg.dc_layers) - 2) if fuse else ()     # fuse_head: layer 0's output, fuse_tail: the last stored one
    for li in fused_layers:
        with pytest.raises(gw.GwError) as e:
            dc.activation(li)
        assert e.value.code == gw.GW_ESTATE
    od, et = util.oracle_dtype(dtype), util.elem_tol(dtype)
    n_up = 8
    x = synth.multi_stream(3, cfg.stream, n_up * 512)
    xd = _dev(x)
    for t in range(n_up):
        st.update(xd[:, :, t * 512:(t + 1) * 512].contiguous())
        dc.forward()
        dc.cleaned(gw.GW_FINAL)
    prepared = [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.dc_layers, dc_params2[0])]
    for i in range(2):
        snap, _ = oracle.snapshot(x[i], n_up - 1, 512, 4096)
        ref_p, acts = oracle.deepclean_forward(snap[cfg.stream.witness_rows(0)].astype(np.float64), cfg.dc_layers,
                                               prepared, return_all=True)
        for li, (layer, ref) in enumerate(zip(cfg.dc_layers[:-1], acts[:-1])):
            if li in fused_layers:
                continue
            got = dc.activation(li).float().cpu().numpy()[i, 0]          # [L][Cp]
            assert got.shape[0] == ref.shape[1]
            assert np.all(got[:, layer.cout:] == 0.0), "padded channels must stay zero"
            # internal activations carry their own storage rounding on top of the propagated error; an
            # indexing bug would be O(1), so bf16 layers get a loose per-element bar here (outputs: `et`)
            util.check_network_output(got[:, :layer.cout].T, ref, f"layer {li} stream {i}",
                                      elem=1e-1 if dtype == gw.GW_BF16 else et)
        pred = dc.noise().cpu().numpy()[i, 0]
        util.check_network_output(pred, ref_p, f"prediction stream {i}", elem=et)
        # Against the storage-rounded oracle what is left is implementation error only (fp32 accumulation order,
        # hardware tanh, the rounding flips they cause): the storage-format floor argument does not apply here, so
        # BOTH dtypes are held to north_star's per-element bar (2e-2 RMS) and to a 3e-3 relative-L2 bar.
        xin = snap[cfg.stream.witness_rows(0)].astype(np.float64)
        ref_r, acts_r = oracle.deepclean_forward(xin, cfg.dc_layers, prepared, act_dtype=od, return_all=True)
        r = util.check_network_output(pred, ref_r, f"prediction vs storage-rounded oracle, stream {i}",
                                      elem=util.ELEM_RMS, rel_l2=3e-3)
        worst_layer = 0.0
        for li, (layer, ref) in enumerate(zip(cfg.dc_layers[:-1], acts_r[:-1])):
            if li in fused_layers:
                continue
            got = dc.activation(li).float().cpu().numpy()[i, 0]
            # stored 16-bit values: a rounding that flips costs one unit in the last place of the value's binade (bf16:
            # 2^-8 = 3.9e-3 for |v| in [0.5, 1), i.e. ~1.3e-2 of a layer RMS of 0.3), and flips propagate; the bar for
            # the STORED layers is therefore two such units (bf16 4e-2 RMS, fp16 5e-3 RMS), still 2.5x tighter than the
            # 1e-1 used against the unrounded oracle above; the fp32 prediction itself is held to 2e-2 RMS.
            _, wl = util.check_network_output(got[:, :layer.cout].T, ref, f"layer {li} vs storage-rounded oracle, stream {i}",
                                              elem=4e-2 if dtype == gw.GW_BF16 else 5e-3, rel_l2=3e-3)
            worst_layer = max(worst_layer, wl)
        # total error against the model with UNROUNDED fp64 weights (reported: weight quantisation is part of the model
        # by reading A9, so this is context, not a bar; only a loose sanity bound is asserted)
        unr = [util.unrounded_conv(l, p) for l, p in zip(cfg.dc_layers, dc_params2[0])]
        ref_u = oracle.deepclean_forward(xin, cfg.dc_layers, unr)
        du = pred - ref_u
        rel_u = float(np.linalg.norm(du) / np.linalg.norm(ref_u))
        worst_u = float(np.max(np.abs(du)) / np.sqrt(np.mean(ref_u ** 2)))
        assert rel_u <= 5e-2
        print(f"dtype {'bf16' if dtype == gw.GW_BF16 else 'fp16'} fuse {fuse} stream {i}: vs storage-rounded oracle rel L2 "
              f"{r[0]:.2e}, worst/RMS {r[1]:.2e} (layers: worst/RMS {worst_layer:.2e}); vs fp64-weight model rel L2 {rel_u:.2e}, "
              f"worst/RMS {worst_u:.2e}")


# ----------------------------------------------------------------------------- classifier (C2)
@pytest.mark.parametrize("fuse", [1, 0])
@pytest.mark.parametrize("length,batch", [(4096, 24), (1024, 5)])
def test_bbh_batch_matches_oracle(length, batch, fuse):
    """fuse = 1: the one-kernel, shared-memory-resident classifier (gw_options.fuse_bbh, the default); 0: three kernels."""
    cfg = S.config_c2()
    cp, dp = util.centred_bbh_params(202, cfg.bbh_convs, cfg.bbh_dense, length)
    bbh = gw.Bbh(None, cfg.bbh_convs, cp, dp, length, gw.GW_BF16, n_det=2, max_batch=32, opts=gw.Options(fuse_bbh=fuse))
    x = synth.bbh_windows(2, batch, length)
    got = bbh.score_batch(_dev(x)).cpu().numpy()
    pc = [oracle.prepare_conv(l, p, oracle.DT_BF16) for l, p in zip(cfg.bbh_convs, cp)]
    pd = [oracle.prepare_dense(p) for p in dp]
    ref = np.array([oracle.bbh_forward(x[i], cfg.bbh_convs, pc, pd) for i in range(batch)])
    assert np.max(np.abs(got - ref)) <= util.SCORE_ABS, (got, ref)
    assert np.max(np.abs(util.logit(got) - util.logit(ref))) <= util.LOGIT_ABS, (got, ref)
    assert 0.2 < np.mean(ref) < 0.8 and np.std(ref) > 1e-2, "scores should not be degenerate"
    print("bbh scores: max |d| %.2e, max |d logit| %.2e, ref range %.3f..%.3f" % (
        np.max(np.abs(got - ref)), np.max(np.abs(util.logit(got) - util.logit(ref))), ref.min(), ref.max()))


@pytest.mark.parametrize("dtype", [gw.GW_FP16, gw.GW_BF16])
@pytest.mark.parametrize("length,n_det,scale,white", [(512, 2, 1.0, False), (2048, 1, 1.0, True), (1536, 2, 2.0 ** -12, False),
                                                     (4096, 2, 2.0 ** 17, True), (3584, 2, 1.0, False)])
def test_bbh_fused_kernel_shapes_scales_and_whitening(length, n_det, scale, white, dtype):
    """The one-kernel classifier at every window length it accepts (tile counts 1..8, one and two block-2 tiles), with one
    detector, with D12 whitening (64 taps: the longest history), and with inputs far outside fp16 range in either direction
    (its first block feeds the tensor core a power-of-two-scaled (hi, lo) pair per sample): against the oracle, and
    against the three-kernel path, which computes the first block in fp32 on CUDA cores."""
    convs = S.bbh_layers((n_det, 32, 64, 128))
    dense = (128, 64, 1)
    od = oracle.DT_BF16 if dtype == gw.GW_BF16 else oracle.DT_FP16
    rng = np.random.default_rng(length + n_det)
    g = None
    if white:
        g = (rng.standard_normal((n_det, 64)) * np.exp(-np.arange(64) / 6.0)).astype(np.float32)
        g[:, 0] = 1.0
    x = (synth.bbh_windows(7, 6, length)[:, :n_det] * scale).astype(np.float32)
    xw = x if g is None else np.stack([np.stack([oracle.fir_causal(x[i][d], g[d]) for d in range(n_det)]) for i in range(len(x))])
    # centre the logits on THESE inputs (weights of the first block absorb the input scale)
    cp, dp = synth.bbh_params(303, convs, dense)
    cp[0]["w"] = (cp[0]["w"] / np.float32(scale)).astype(np.float32)
    pc = [oracle.prepare_conv(l, p, od) for l, p in zip(convs, cp)]
    mean_logit = float(np.mean([oracle.bbh_forward(xw[i], convs, pc, [oracle.prepare_dense(p) for p in dp], return_logit=True)
                                for i in range(len(x))]))
    dp[-1]["b"] = (dp[-1]["b"] - np.float32(mean_logit)).astype(np.float32)
    pd = [oracle.prepare_dense(p) for p in dp]
    ref = np.array([oracle.bbh_forward(xw[i], convs, pc, pd) for i in range(len(x))])
    got = {}
    for fuse in (1, 0):
        bbh = gw.Bbh(None, convs, cp, dp, length, dtype, n_det=n_det, max_batch=8, opts=gw.Options(fuse_bbh=fuse))
        if g is not None:
            bbh.set_whitening(g)
        got[fuse] = bbh.score_batch(_dev(x)).cpu().numpy()
        assert np.max(np.abs(got[fuse] - ref)) <= util.SCORE_ABS, (fuse, got[fuse], ref)
        assert np.max(np.abs(util.logit(got[fuse]) - util.logit(ref))) <= util.LOGIT_ABS, (fuse, got[fuse], ref)
    assert np.std(ref) > 1e-3, "scores should not be degenerate"
    print("fused classifier L=%d D=%d scale=%g white=%s: max |d| vs oracle %.2e (three kernels %.2e), fused vs three kernels %.2e" % (
        length, n_det, scale, white, np.max(np.abs(got[1] - ref)), np.max(np.abs(got[0] - ref)), np.max(np.abs(got[1] - got[0]))))


# -------------------------------------------------------------------- end-to-end small ensemble
@pytest.mark.parametrize("dtype", [gw.GW_BF16, gw.GW_FP16])
def test_small_ensemble_eager_matches_oracle(dtype):
    cfg = S.config_small_ensemble(2)
    stats = _run_streaming(cfg, dtype, cfg.n_updates, white=False)
    print("ensemble worst:", stats)


def test_small_ensemble_graph_matches_oracle_and_eager():
    cfg = S.config_small_ensemble(2)
    _run_streaming(cfg, gw.GW_BF16, cfg.n_updates, white=False, use_graph=True)


@pytest.mark.parametrize("agg", [S.AGG_HANN_OLA, S.AGG_LAST_STRIDE])
@pytest.mark.parametrize("delta", [256, 788, 131])
def test_small_ensemble_latency_offset_scores_match_oracle(agg, delta):
    """D8 with delta > 0 WITH the classifier attached: the window the classifier scores ends `delta`
    samples before the newest sample (delta = S, 3S + 20, and 131: not a multiple of 4, which takes the scalar
    aggregation kernel).  Scores, running estimate and running cleaned strain against the oracle, both aggregation
    modes; the oracle's own window arithmetic is pinned by direct slicing in tests/test_oracle_pins.py."""
    cfg = S.config_small_ensemble(2)
    assert cfg.bbh_len + delta <= cfg.stream.window
    stats = _run_streaming(cfg, gw.GW_FP16, cfg.n_updates, white=False, agg=agg, delta=delta)
    print(f"delta={delta} agg={agg}: worst", stats)


def test_small_ensemble_latency_offset_through_the_graph():
    """The same through gw_step (the captured graph bakes delta into the aggregation node)."""
    cfg = S.config_small_ensemble(2)
    _run_streaming(cfg, gw.GW_FP16, cfg.n_updates, white=False, agg=S.AGG_HANN_OLA, delta=512, use_graph=True)
    _run_streaming(cfg, gw.GW_FP16, cfg.n_updates, white=False, agg=S.AGG_LAST_STRIDE, delta=256, use_graph=True)


# ------------------------------------------------ D11 / D12: band-limited emitted estimate, whitened classifier input
@pytest.mark.parametrize("agg,delta,incremental", [(S.AGG_HANN_OLA, 0, False), (S.AGG_LAST_STRIDE, 256, False),
                                                   (S.AGG_HANN_OLA, 0, True)])
def test_postfilter_and_whitening_match_oracle(agg, delta, incremental):
    """DESIGN.md D11: a causal FIR over the STREAM of emitted estimate samples, state carried from
    update to update; D12: FIR whitening of the classifier window.  Final cleaned samples (through the
    graph) and scores against the oracle; the identity filters are bit-exact no-ops; running values stay unfiltered."""
    cfg = S.config_small_ensemble(2)
    sp = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    n_up = 14
    rng = np.random.default_rng(77)
    h = (0.3 * rng.standard_normal(17)).astype(np.float32)
    g = (0.2 * rng.standard_normal((sp.n_det, 12))).astype(np.float32)
    g[:, 0] += 1.0
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    xc = torch.from_numpy(np.ascontiguousarray(x.reshape(sp.n_streams, sp.channels, n_up, sp.stride).transpose(2, 0, 1, 3))).cuda()
    dtype = gw.GW_FP16
    outs = {}
    for name, pf, wh in (("none", None, None), ("ident", np.ones(1, np.float32), np.ones((sp.n_det, 1), np.float32)), ("filt", h, g)):
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, agg, delta, gw.Options(incremental=incremental))
        if pf is not None:
            dc.set_postfilter(pf)
            bbh.set_whitening(wh)
        cs = torch.cuda.Stream()
        sc = torch.zeros(sp.n_streams, device="cuda")
        fin = torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda")
        torch.cuda.synchronize()
        res = []
        for t in range(n_up):
            pipe.step(xc[t], sc, fin, cs)
            cs.synchronize()
            res.append((fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
        outs[name] = res
        if name == "filt":
            with pytest.raises(gw.GwError) as e:
                dc.set_postfilter(h)                        # after the first update: the filter carries state
            assert e.value.code == gw.GW_ESTATE
    for t in range(n_up):
        assert np.array_equal(outs["none"][t][0], outs["ident"][t][0]) and np.array_equal(outs["none"][t][1], outs["ident"][t][1]), t
    oracles = [util.make_stream_oracle(cfg, dc_params, bbh_params, dtype, n_up, agg, delta) for _ in range(sp.n_streams)]
    for o in oracles:
        o.postfilter = np.asarray(h, np.float64)
        o.whiten = np.asarray(g, np.float64)
    worst = 0.0
    differs = False
    for t in range(n_up):
        fin_t, sc_t = outs["filt"][t]
        differs = differs or not np.array_equal(fin_t, outs["none"][t][0])
        for i, orc in enumerate(oracles):
            ref = orc.update(x[i][:, t * sp.stride:(t + 1) * sp.stride])
            for d in range(sp.n_det):
                _, w = util.check_network_output(fin_t[i, d], ref["cleaned_final"][d], f"post-filtered final update {t} stream {i} det {d}",
                                                 rms_ref=ref["pred"][d])
                worst = max(worst, w)
            assert abs(float(sc_t[i]) - ref["score"]) <= util.SCORE_ABS, (t, i, float(sc_t[i]), ref["score"])
            assert abs(util.logit(sc_t[i]) - util.logit(ref["score"])) <= util.LOGIT_ABS, (t, i, float(sc_t[i]), ref["score"])
    assert differs, "the filters must change something"
    print(f"D11/D12 agg={agg} delta={delta} incremental={incremental}: worst |d final|/RMS(pred) {worst:.3e}")


def test_whitened_batch_classifier_and_filter_argument_checks():
    cfg = S.config_c2()
    L, batch = 1024, 6
    cp, dp = util.centred_bbh_params(202, cfg.bbh_convs, cfg.bbh_dense, L)
    bbh = gw.Bbh(None, cfg.bbh_convs, cp, dp, L, gw.GW_BF16, n_det=2, max_batch=8)
    x = synth.bbh_windows(2, batch, L)
    g = np.array([[1.0, -0.6, 0.25, 0.0, 0.1], [0.9, 0.3, -0.2, 0.05, 0.0]], np.float32)
    bbh.set_whitening(g)
    got = bbh.score_batch(_dev(x)).cpu().numpy()
    pc = [oracle.prepare_conv(l, p, oracle.DT_BF16) for l, p in zip(cfg.bbh_convs, cp)]
    pd = [oracle.prepare_dense(p) for p in dp]
    ref = np.array([oracle.bbh_forward(np.stack([oracle.fir_causal(x[i][d], g[d]) for d in range(2)]), cfg.bbh_convs, pc, pd)
                    for i in range(batch)])
    assert np.max(np.abs(got - ref)) <= util.SCORE_ABS, (got, ref)
    assert np.max(np.abs(util.logit(got) - util.logit(ref))) <= util.LOGIT_ABS, (got, ref)
    bbh.set_whitening(None)
    plain = bbh.score_batch(_dev(x)).cpu().numpy()
    assert not np.array_equal(plain, got)
    with pytest.raises(gw.GwError):
        bbh.set_whitening(np.ones((2, 65), np.float32))      # more than 64 taps
    c0 = S.config_c0()
    st = gw.Stream(c0.stream)
    dc = gw.DeepClean(st, c0.dc_layers, util.make_params(c0)[0], gw.GW_FP16)
    with pytest.raises(gw.GwError):
        dc.set_postfilter(np.ones(66, np.float32))           # n_taps - 1 > stride (64) and > 64 taps
    with pytest.raises(gw.GwError):
        dc.set_postfilter(np.array([1.0, np.nan], np.float32))


# ------------------------------------------------ D13 incremental path (gw_options.incremental)
@pytest.mark.parametrize("W,S_,n,dtype", [(2048, 256, 3, gw.GW_FP16), (8192, 512, 2, gw.GW_BF16), (32768, 512, 2, gw.GW_FP16),
                                          (4096, 16, 1, gw.GW_FP16), (32768, 1024, 1, gw.GW_BF16), (32768, 256, 1, gw.GW_FP16),
                                          (8192, 1024, 6, gw.GW_FP16), (16384, 256, 4, gw.GW_BF16), (8192, 256, 8, gw.GW_FP16)])
def test_incremental_path_is_bit_identical_to_full_recompute(W, S_, n, dtype):
    """DESIGN.md D13: with gw_options.incremental every layer's activations live in rings
    over absolute position and an update recomputes only the rows near the two window edges (tests/test_oracle_pins.py
    pins which).  The result must be the SAME NUMBERS as full recomputation: raw prediction, final cleaned samples and
    scores compared with array_equal over more than 2 W/S updates, warm-up included (the first update fills the rings
    with whole windows), through the CUDA graph; the stored activations of every layer as well at the end.
    Even stream counts take the CTA-pair layers' packed form (both zones of one, two or four windows in one tile: stride
    1024 / 512 / 256 with stream counts that divide), odd ones the tile-per-zone form."""
    cfg0 = S.config_c3(n, S_, W)
    Lb = min(4096, W // 2)
    cfg = S.Config("inc", cfg0.stream, cfg0.dc_layers, cfg0.bbh_convs, cfg0.bbh_dense, Lb, 0, 11)
    sp = cfg.stream
    k = W // S_
    n_up = min(2 * k + 5, 300)
    dc_params, bbh_params = util.make_params(cfg)
    x = synth.multi_stream(cfg.seed, sp, n_up * S_)
    xc = torch.from_numpy(np.ascontiguousarray(x.reshape(n, sp.channels, n_up, S_).transpose(2, 0, 1, 3))).cuda()
    outs, acts = {}, {}
    for inc in (0, 1):
        # fuse_head = 0: the whole-window engine stores layer 0's output, so that every layer can be compared
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, opts=gw.Options(incremental=inc, fuse_head=0))
        cs = torch.cuda.Stream()
        sc = torch.zeros(n, device="cuda")
        fin = torch.zeros((n, sp.n_det, S_), device="cuda")
        torch.cuda.synchronize()
        res = []
        for t in range(n_up):
            pipe.step(xc[t], sc, fin, cs)
            cs.synchronize()
            if t < 4 or t % 7 == 0 or t >= n_up - 3:
                res.append((t, dc.noise().cpu().numpy(), fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
        outs[inc] = res
        acts[inc] = [dc.activation(li).cpu().view(torch.int16).numpy() for li in range(-1, len(cfg.dc_layers) - 2)]
        if inc:
            assert pipe.graph_nodes() == outs_nodes, "same kernels per step either way"
        else:
            outs_nodes = pipe.graph_nodes()
    for (t, p0, f0, s0), (_, p1, f1, s1) in zip(outs[0], outs[1]):
        assert np.array_equal(p0, p1), ("pred", t, np.argwhere(p0 != p1)[:4])
        assert np.array_equal(f0, f1), ("final", t)
        assert np.array_equal(s0, s1), ("scores", t)
    for li, (a0, a1) in enumerate(zip(acts[0], acts[1])):
        assert np.array_equal(a0, a1), ("activation after layer", li - 1)


@pytest.mark.parametrize("dtype", [gw.GW_FP16, gw.GW_BF16])
def test_incremental_path_matches_oracle_eager_and_graph(dtype):
    """The oracle parity suite of the small ensemble with the incremental path switched on (the oracle is unchanged:
    it recomputes every window from scratch)."""
    cfg = S.config_small_ensemble(2)
    _run_streaming(cfg, dtype, cfg.n_updates, white=False, incremental=True)
    _run_streaming(cfg, dtype, cfg.n_updates, white=False, incremental=True, use_graph=True)
    _run_streaming(cfg, dtype, cfg.n_updates, white=False, incremental=True, agg=S.AGG_LAST_STRIDE, delta=256)


def test_incremental_path_rejects_shapes_it_cannot_serve():
    cfg = S.config_c0()                                  # W = 512: not a multiple of 128 * 2^3
    dc_params, _ = util.make_params(cfg)
    st = gw.Stream(cfg.stream)
    with pytest.raises(gw.GwError) as e:
        gw.DeepClean(st, cfg.dc_layers, dc_params, gw.GW_FP16, opts=gw.Options(incremental=1))
    assert e.value.code == gw.GW_EINVAL and "incremental" in str(e.value)
    cfg2 = S.Config("odd", S.StreamSpec(1, 2, 4096, 2048, 200), S.config_c1().dc_layers, seed=1)   # 200 % 16 != 0
    st2 = gw.Stream(cfg2.stream)
    with pytest.raises(gw.GwError):
        gw.DeepClean(st2, cfg2.dc_layers, [synth.deepclean_params(d, cfg2.dc_layers) for d in range(2)], gw.GW_FP16,
                     agg=S.AGG_LAST_STRIDE, opts=gw.Options(incremental=1))
    with pytest.raises(gw.GwError):
        gw.DeepClean(st2, cfg2.dc_layers, [synth.deepclean_params(d, cfg2.dc_layers) for d in range(2)], gw.GW_FP16,
                     agg=S.AGG_LAST_STRIDE, opts=gw.Options(incremental=1, conv_impl=gw.GW_IMPL_SIMT))


def test_results_do_not_depend_on_batching():
    """updates are serial per stream, streams are independent: stream i's results are
    bit-identical whether it runs alone or batched with others."""
    cfg2 = S.config_small_ensemble(3)
    dc_params, bbh_params = util.make_params(cfg2)
    x = synth.multi_stream(cfg2.seed, cfg2.stream, 6 * cfg2.stream.stride)
    outs = {}
    for which in ("all", 0, 2):
        if which == "all":
            cfg, xs = cfg2, x
        else:
            cfg, xs = S.config_small_ensemble(1), x[which:which + 1]
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, gw.GW_BF16)
        xd = _dev(xs)
        res = []
        for t in range(6):
            stream.update(xd[:, :, t * cfg.stream.stride:(t + 1) * cfg.stream.stride].contiguous())
            dc.forward()
            res.append((dc.cleaned(gw.GW_FINAL).cpu().numpy(), bbh.score().cpu().numpy()))
        outs[which] = res
    for which in (0, 2):
        for t in range(6):
            assert np.array_equal(outs["all"][t][0][which], outs[which][t][0][0])
            assert outs["all"][t][1][which] == outs[which][t][1][0]


def test_zero_network_returns_strain_bit_exact():
    cfg = S.config_c0()
    zero = [[{"w": np.zeros(l.wshape(), np.float32), "b": np.zeros(l.cout, np.float32)} for l in cfg.dc_layers]]
    st = gw.Stream(cfg.stream)
    dc = gw.DeepClean(st, cfg.dc_layers, zero, gw.GW_BF16)
    x = synth.multi_stream(9, cfg.stream, 12 * 64, white=True)
    xd = _dev(x)
    for t in range(12):
        st.update(xd[:, :, t * 64:(t + 1) * 64].contiguous())
        dc.forward()
        run = dc.cleaned(gw.GW_RUNNING).cpu().numpy()[0, 0]
        first = (t + 1) * 64 - 512
        lo = max(first, 0)
        exp = x[0, cfg.stream.strain_row(0), lo:first + 512]
        assert np.array_equal(run[lo - first:].view(np.uint32), exp.view(np.uint32))
        assert np.all(run[:lo - first] == 0.0)


def test_call_order_is_enforced():
    cfg = S.config_c0()
    dc_params, _ = util.make_params(cfg)
    st = gw.Stream(cfg.stream)
    dc = gw.DeepClean(st, cfg.dc_layers, dc_params, gw.GW_BF16)
    new = torch.zeros((1, 22, 64), device="cuda")
    with pytest.raises(gw.GwError) as e:
        dc.forward()
    assert e.value.code == gw.GW_ESTATE
    st.update(new)
    with pytest.raises(gw.GwError) as e:
        st.update(new)
    assert e.value.code == gw.GW_ESTATE
    with pytest.raises(gw.GwError) as e:
        dc.cleaned()
    assert e.value.code == gw.GW_ESTATE
    dc.forward()
    with pytest.raises(gw.GwError) as e:
        dc.forward()
    assert e.value.code == gw.GW_ESTATE
    dc.cleaned()
    with pytest.raises(gw.GwError) as e:
        dc.cleaned()
    assert e.value.code == gw.GW_ESTATE
    st.update(new)


# ------------------------------------------------- full size: the launch configuration bench.py times
@pytest.mark.gpu
@pytest.mark.parametrize("dtype,n,full_chain,incremental", [(gw.GW_FP16, 128, True, False), (gw.GW_BF16, 128, False, False),
                                                           (gw.GW_FP16, 512, False, False), (gw.GW_FP16, 128, False, True)])
def test_full_size_c4_sampled_streams_match_oracle(dtype, n, full_chain, incremental):
    """BASELINE.json configs[4] as bench.py runs it: n = 128 (and 512) streams x 2 detectors, W = 32768, S = 512, one
    CUDA-graph launch per stride -- every CTA of the persistent conv GEMMs walks many tiles, weight blocks stream
    through the pair-mode ring, both MMA warps and PDL are live -- compared with the oracle on FULLY POPULATED windows:
    the engine is pre-rolled through W/S = 64 updates (the sampled oracles only record those samples, oracle.skip), then
    the raw predictions of three sampled streams (first, middle, last) are checked on 3 further updates.  With
    full_chain (n = 128, fp16) the oracle of stream 0 is run through ALL 72 updates instead, so that its overlap-add
    state is complete: final cleaned samples and classifier scores are then checked on the 8 steady-state updates as
    well as on the warm-up ones.  A property that holds at any size covers the unsampled streams: streams fed identical
    samples give bit-identical results wherever they sit in the batch."""
    cfg = S.config_c3(n, 512, 32768)
    sp = cfg.stream
    k = sp.window // sp.stride
    n_cmp = 8 if full_chain else 3
    n_up = k + n_cmp
    dc_params, bbh_params = util.make_params(cfg)
    one = S.StreamSpec(1, sp.n_det, sp.fs, sp.window, sp.stride, sp.n_witness)
    base = np.stack([synth.stream_channels(cfg.seed + i, one, n_up * sp.stride) for i in range(3)])
    sampled = {0: 0, 77: 1, n - 1: 2}                    # stream index -> which base signal it carries
    which = np.array([sampled.get(i, i % 3) for i in range(n)])
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, opts=gw.Options(incremental=incremental))
    oracles = {i: util.make_stream_oracle(S.config_c3(1, 512, 32768), dc_params, bbh_params, dtype, n_up) for i in sampled}
    base_d = _dev(base)
    which_d = torch.from_numpy(which).cuda()
    cs = torch.cuda.Stream()
    scores_d = torch.zeros(n, device="cuda")
    final_d = torch.zeros((n, sp.n_det, sp.stride), device="cuda")
    et = util.elem_tol(dtype)
    worst = {"pred": 0.0, "final": 0.0, "score": 0.0}
    for t in range(n_up):
        new = base_d[:, :, t * sp.stride:(t + 1) * sp.stride][which_d].contiguous()     # [n][C][S]
        cs.wait_stream(torch.cuda.current_stream())
        pipe.step(new, scores_d, final_d, cs)
        cs.synchronize()
        compare_all = t >= k
        for i, orc in oracles.items():
            xs = base[sampled[i]][:, t * sp.stride:(t + 1) * sp.stride]
            chain = full_chain and i == 0
            if not compare_all and not chain:
                orc.skip(xs)                             # zero oracle cost: only records the samples
        if not compare_all and not full_chain:
            continue
        pred = dc.noise().cpu().numpy()
        final = final_d.cpu().numpy()
        scores = scores_d.cpu().numpy()
        for i, orc in oracles.items():
            chain = full_chain and i == 0
            if not compare_all and not chain:
                continue
            if chain and not compare_all and t % 8 != 7 and t > 2:
                orc.update(base[sampled[i]][:, t * sp.stride:(t + 1) * sp.stride])   # state only (warm-up updates are sampled)
                continue
            ref = orc.update(base[sampled[i]][:, t * sp.stride:(t + 1) * sp.stride])
            for d in range(sp.n_det):
                tag = f"full size update {t} stream {i} det {d}"
                _, w1 = util.check_network_output(pred[i, d], ref["pred"][d], "pred " + tag, elem=et)
                worst["pred"] = max(worst["pred"], w1)
                if chain:                                # overlap-add state complete: finals and scores are meaningful
                    _, w2 = util.check_network_output(final[i, d], ref["cleaned_final"][d], "final " + tag, rms_ref=ref["pred"][d], elem=et)
                    worst["final"] = max(worst["final"], w2)
            if chain:
                assert abs(float(scores[i]) - ref["score"]) <= util.SCORE_ABS, (t, i, float(scores[i]), ref["score"])
                worst["score"] = max(worst["score"], abs(float(scores[i]) - ref["score"]))
        if compare_all:
            for i in range(n):                           # position in the batch does not matter
                j = {0: 0, 1: 77, 2: n - 1}[which[i]]
                assert np.array_equal(pred[i], pred[j]), (t, i, j)
                assert np.array_equal(final[i], final[j]) and scores[i] == scores[j], (t, i, j)
    print(f"full size n={n} dtype={'bf16' if dtype == gw.GW_BF16 else 'fp16'}{' incremental' if incremental else ''}: fully populated windows, worst |d|/RMS "
          f"pred {worst['pred']:.3e} final {worst['final']:.3e}, worst |d score| {worst['score']:.2e}")


@pytest.mark.gpu
def test_host_step_async_equals_device_step_bitwise():
    """gw_step_host_async (double-buffered input staging on an internal copy stream) and gw_step_host deliver
    exactly what gw_step computes from device-resident inputs."""
    cfg = S.config_small_ensemble(3)
    sp = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    n_up = 7
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    outs = {}
    for mode in ("device", "host", "async"):
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, gw.GW_FP16)
        cs = torch.cuda.Stream()
        res = []
        if mode == "device":
            xd = _dev(x)
            sc = torch.zeros(sp.n_streams, device="cuda")
            fin = torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda")
            for t in range(n_up):
                new = xd[:, :, t * sp.stride:(t + 1) * sp.stride].contiguous()
                cs.wait_stream(torch.cuda.current_stream())
                pipe.step(new, sc, fin, cs)
                cs.synchronize()
                res.append((fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
        else:
            xin = [torch.from_numpy(np.ascontiguousarray(x[:, :, t * sp.stride:(t + 1) * sp.stride])).pin_memory() for t in range(n_up)]
            sch = [torch.zeros(sp.n_streams).pin_memory() for _ in range(n_up)]
            finh = [torch.zeros((sp.n_streams, sp.n_det, sp.stride)).pin_memory() for _ in range(n_up)]
            for t in range(n_up):
                (pipe.step_host if mode == "host" else pipe.step_host_async)(xin[t], sch[t], finh[t], cs)
            cs.synchronize()
            res = [(finh[t].numpy().copy(), sch[t].numpy().copy()) for t in range(n_up)]
        outs[mode] = res
    for mode in ("host", "async"):
        for t in range(n_up):
            assert np.array_equal(outs[mode][t][0], outs["device"][t][0]), (mode, t)
            assert np.array_equal(outs[mode][t][1], outs["device"][t][1]), (mode, t)


# --------------------------------------------------------------- offline / non-streaming mode (D9)
@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [gw.GW_FP16, gw.GW_BF16])
def test_offline_matches_oracle_and_streaming_finals(dtype):
    """B windows of one stream per launch: against the fp64 offline oracle (north_star tolerances on the raw
    predictions and on the estimate), and -- a property that needs no oracle -- every sample covered by all W/S
    windows is BIT-identical to the final value the streaming path emits for it."""
    cfg = S.config_small_ensemble(1)                     # W = 2048, S = 256, k = 8, two detectors
    sp = cfg.stream
    W, St = sp.window, sp.stride
    k = W // St
    B = 21                                               # several tiles per window, odd count, ragged coverage at both ends
    T = W + (B - 1) * St
    dc_params, _ = util.make_params(cfg)
    x = synth.stream_channels(cfg.seed + 40, sp, T)
    off = gw.Offline(sp, cfg.dc_layers, dc_params, B, dtype)
    assert off.samples == T
    cleaned, noise = off.run(_dev(x))
    torch.cuda.synchronize()
    cleaned, noise, pred = cleaned.cpu().numpy(), noise.cpu().numpy(), off.predictions().cpu().numpy()
    od = util.oracle_dtype(dtype)
    rows = [(sp.witness_rows(d), sp.strain_row(d)) for d in range(sp.n_det)]
    odc = [(cfg.dc_layers, [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.dc_layers, dc_params[d])]) for d in range(sp.n_det)]
    ref = oracle.offline_clean(x, W, St, rows, odc)
    et = util.elem_tol(dtype)
    for d in range(sp.n_det):
        for j in (0, 1, B // 2, B - 1):
            util.check_network_output(pred[j, d], ref["pred"][d, j], f"offline pred window {j} det {d}", elem=et)
        rms_ref = ref["pred"][d]
        util.check_network_output(noise[d], ref["nhat"][d], f"offline nhat det {d}", rms_ref=rms_ref, elem=et)
        util.check_network_output(cleaned[d], ref["cleaned"][d], f"offline cleaned det {d}", rms_ref=rms_ref, elem=et)
        assert noise[d, 0] == 0.0 and cleaned[d, 0] == x[sp.strain_row(d), 0]
    # the streaming path over the same samples
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, None, dtype)
    xd = _dev(x[None])
    finals = np.full((sp.n_det, T), np.nan, dtype=np.float32)
    for t in range(T // St):
        stream.update(xd[:, :, t * St:(t + 1) * St].contiguous())
        dc.forward()
        f = dc.cleaned(gw.GW_FINAL).cpu().numpy()[0]
        a0 = (t + 1) * St - W
        if a0 >= 0:
            finals[:, a0:a0 + St] = f
    lo, hi = (k - 1) * St, T - (k - 1) * St
    assert hi - lo >= 2 * St
    assert np.array_equal(cleaned[:, lo:hi], finals[:, lo:hi])


# ------------------------------------------------------- pre/post-processing (reading A14)
def _scaling_for(sp, seed=0):
    rng = np.random.default_rng(900 + seed)
    return (rng.normal(0, 0.5, (sp.n_det, sp.n_witness)).astype(np.float32),
            rng.uniform(0.5, 2.0, (sp.n_det, sp.n_witness)).astype(np.float32),
            rng.normal(0, 0.3, sp.n_det).astype(np.float32), rng.uniform(0.5, 2.0, sp.n_det).astype(np.float32))


@pytest.mark.gpu
@pytest.mark.parametrize("stride", [256, 255])           # mirror-ring path / gather path (odd stride)
def test_scaled_streaming_matches_oracle(stride):
    cfg0 = S.config_small_ensemble(2)
    sp = S.StreamSpec(2, 2, 4096, 2048, stride)          # 255 does not divide 2048: LAST_STRIDE aggregation there
    cfg = S.Config("scaled", sp, cfg0.dc_layers, cfg0.bbh_convs, cfg0.bbh_dense, cfg0.bbh_len, 10, 5)
    dtype = gw.GW_FP16
    agg = S.AGG_HANN_OLA if stride == 256 else S.AGG_LAST_STRIDE
    dc_params, bbh_params = util.make_params(cfg)
    scaling = _scaling_for(sp)
    n_up = 10
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, agg, 0)
    dc.set_scaling(*scaling)
    oracles = [util.make_stream_oracle(cfg, dc_params, bbh_params, dtype, n_up, agg, 0, scaling=scaling) for _ in range(sp.n_streams)]
    xd = _dev(x)
    for t in range(n_up):
        stream.update(xd[:, :, t * sp.stride:(t + 1) * sp.stride].contiguous())
        dc.forward()
        pred = dc.noise().cpu().numpy()
        running = dc.cleaned(gw.GW_RUNNING).cpu().numpy()
        nhat = dc.noise_estimate().cpu().numpy()
        scores = bbh.score().cpu().numpy()
        for i, orc in enumerate(oracles):
            ref = orc.update(x[i][:, t * sp.stride:(t + 1) * sp.stride])
            for d in range(sp.n_det):
                tag = f"scaled update {t} stream {i} det {d}"
                util.check_network_output(pred[i, d], ref["pred"][d], "pred " + tag)
                rms_n = float(scaling[3][d]) * ref["pred"][d]          # the estimate's scale after rescaling
                util.check_network_output(nhat[i, d], ref["nhat_running"][d], "nhat " + tag, rms_ref=rms_n)
                util.check_network_output(running[i, d], ref["cleaned_running"][d], "cleaned " + tag, rms_ref=rms_n)
            assert abs(float(scores[i]) - ref["score"]) <= util.SCORE_ABS
    with pytest.raises(gw.GwError):
        dc.set_scaling(*scaling)                        # after the first update: GW_ESTATE


@pytest.mark.gpu
def test_identity_scaling_is_bit_exact_and_offline_scaling_matches_oracle():
    cfg = S.config_small_ensemble(1)
    sp = cfg.stream
    dc_params, _ = util.make_params(cfg)
    B = 9
    T = sp.window + (B - 1) * sp.stride
    x = synth.stream_channels(77, sp, T)
    outs = []
    for ident in (False, True):
        off = gw.Offline(sp, cfg.dc_layers, dc_params, B, gw.GW_FP16)
        if ident:
            off.set_scaling(np.zeros((sp.n_det, sp.n_witness)), np.ones((sp.n_det, sp.n_witness)), np.zeros(sp.n_det), np.ones(sp.n_det))
        c, n = off.run(_dev(x))
        outs.append((c.cpu().numpy(), n.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    scaling = _scaling_for(sp, 1)
    off = gw.Offline(sp, cfg.dc_layers, dc_params, B, gw.GW_FP16)
    off.set_scaling(*scaling)
    c, n = off.run(_dev(x))
    c, n = c.cpu().numpy(), n.cpu().numpy()
    rows = [(sp.witness_rows(d), sp.strain_row(d)) for d in range(sp.n_det)]
    odc = [(cfg.dc_layers, [oracle.prepare_conv(l, p, oracle.DT_FP16) for l, p in zip(cfg.dc_layers, dc_params[d])]) for d in range(sp.n_det)]
    ref = oracle.offline_clean(x, sp.window, sp.stride, rows, odc, scaling=scaling)
    for d in range(sp.n_det):
        rms_n = float(scaling[3][d]) * ref["pred"][d]
        util.check_network_output(n[d], ref["nhat"][d], f"offline scaled nhat det {d}", rms_ref=rms_n)
        util.check_network_output(c[d], ref["cleaned"][d], f"offline scaled cleaned det {d}", rms_ref=rms_n)


@pytest.mark.gpu
def test_offline_odd_stride_gather_path_matches_oracle():
    """Odd stride: window starts do not fall on position pairs, so the offline first layer cannot read the
    converted segment through the overlapping-window tensor map and every window is gathered instead."""
    sp = S.StreamSpec(1, 1, 512, 120, 15)
    layers = S.config_c0().dc_layers
    params = [synth.deepclean_params(31, layers)]
    B = 13
    T = sp.window + (B - 1) * sp.stride
    x = synth.stream_channels(32, sp, T, white=True)
    off = gw.Offline(sp, layers, params, B, gw.GW_FP16)
    c, n = off.run(_dev(x))
    c, n = c.cpu().numpy(), n.cpu().numpy()
    odc = [(layers, [oracle.prepare_conv(l, p, oracle.DT_FP16) for l, p in zip(layers, params[0])])]
    ref = oracle.offline_clean(x, sp.window, sp.stride, [(sp.witness_rows(0), sp.strain_row(0))], odc)
    util.check_network_output(n[0], ref["nhat"][0], "offline odd-stride nhat", rms_ref=ref["pred"][0])
    util.check_network_output(c[0], ref["cleaned"][0], "offline odd-stride cleaned", rms_ref=ref["pred"][0])


# ------------------------------------------------------------------ C2 at full size, edge cases
@pytest.mark.gpu
def test_c2_full_batch_sampled_windows_match_oracle():
    """BASELINE.json configs[2]: 256 windows x 2 detectors x 4096 samples, bf16.  The oracle scores sampled windows;
    a property covers the rest: a window's score does not depend on its position in the batch (bit-exact)."""
    cfg = S.config_c2()
    L, batch = 4096, 256
    cp, dp = util.centred_bbh_params(202, cfg.bbh_convs, cfg.bbh_dense, L)
    bbh = gw.Bbh(None, cfg.bbh_convs, cp, dp, L, gw.GW_BF16, n_det=2, max_batch=batch)
    x = synth.bbh_windows(2, batch, L)
    got = bbh.score_batch(_dev(x)).cpu().numpy()
    pc = [oracle.prepare_conv(l, p, oracle.DT_BF16) for l, p in zip(cfg.bbh_convs, cp)]
    pd = [oracle.prepare_dense(p) for p in dp]
    for i in (0, 1, 2, 3, 77, 128, 129, 200, 254, 255):
        ref = oracle.bbh_forward(x[i], cfg.bbh_convs, pc, pd)
        assert abs(float(got[i]) - ref) <= util.SCORE_ABS, (i, float(got[i]), ref)
    perm = np.random.default_rng(0).permutation(batch)
    got_p = bbh.score_batch(_dev(x[perm])).cpu().numpy()
    assert np.array_equal(got_p, got[perm])
    with pytest.raises(gw.GwError):
        bbh.score_batch(_dev(x[:0]))                    # empty batch: GW_EINVAL, nothing launched
    one = bbh.score_batch(_dev(x[5:6])).cpu().numpy()   # batch of one
    assert one[0] == got[5]


@pytest.mark.gpu
def test_degenerate_shapes():
    """Stride = window (no overlap: LAST_STRIDE keeps the whole prediction), a single offline window (the estimate
    is the prediction itself wherever the Hann weight is positive), and a single stream / single detector."""
    layers = S.config_c0().dc_layers
    params = [synth.deepclean_params(61, layers)]
    od = [(layers, [oracle.prepare_conv(l, p, oracle.DT_FP16) for l, p in zip(layers, params[0])])]
    # stride == window
    sp = S.StreamSpec(1, 1, 512, 128, 128)
    cfg = S.Config("k1", sp, layers, seed=8)
    n_up = 4
    x = synth.multi_stream(8, sp, n_up * sp.stride, white=True)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, params, None, gw.GW_FP16, S.AGG_LAST_STRIDE, 0)
    orc = oracle.StreamOracle(sp.channels, sp.window, sp.stride, [(sp.witness_rows(0), sp.strain_row(0))], od, None,
                              agg=oracle.AGG_LAST_STRIDE, max_updates=n_up)
    xd = _dev(x)
    for t in range(n_up):
        stream.update(xd[:, :, t * sp.stride:(t + 1) * sp.stride].contiguous())
        dc.forward()
        fin = dc.cleaned(gw.GW_FINAL).cpu().numpy()[0, 0]
        ref = orc.update(x[0][:, t * sp.stride:(t + 1) * sp.stride])
        util.check_network_output(fin, ref["cleaned_final"][0], f"k=1 final update {t}", rms_ref=ref["pred"][0])
    with pytest.raises(gw.GwError):                     # Hann overlap-add needs at least two windows over a sample
        gw.build_ensemble(cfg, params, None, gw.GW_FP16, S.AGG_HANN_OLA, 0)
    # one offline window
    sp1 = S.StreamSpec(1, 1, 512, 128, 64)
    x1 = synth.stream_channels(9, sp1, sp1.window, white=True)
    off = gw.Offline(sp1, layers, params, 1, gw.GW_FP16)
    c, n = off.run(_dev(x1))
    p = off.predictions().cpu().numpy()[0, 0]
    n = n.cpu().numpy()[0]
    assert n[0] == 0.0
    assert np.allclose(n[1:], p[1:], rtol=2e-6, atol=1e-7)      # w p / w, one rounding each way
    ref = oracle.offline_clean(x1, sp1.window, sp1.stride, [(sp1.witness_rows(0), sp1.strain_row(0))], od)
    util.check_network_output(c.cpu().numpy()[0], ref["cleaned"][0], "single offline window", rms_ref=ref["pred"][0])


@pytest.mark.gpu
def test_c0_against_the_stored_oracle_values():
    """The CUDA path against tests/golden/c0_oracle.txt (values written by the oracle alone, BASELINE.json
    configs[0], fp16): the same bars as the live comparison, on numbers that cannot drift with the code under test."""
    import os
    recs = []
    for line in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c0_oracle.txt")):
        if not line.startswith("#") and line.strip():
            k, t, i, v = line.split()
            recs.append((k, int(t), int(i), float(v)))
    cfg = S.config_c0()
    sp = cfg.stream
    params = [synth.deepclean_params(cfg.seed * 100, cfg.dc_layers)]
    x = synth.multi_stream(cfg.seed, sp, cfg.n_updates * sp.stride, white=True)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, params, None, gw.GW_FP16)
    xd = _dev(x)
    got = {}
    rms = {}
    for t in range(cfg.n_updates):
        stream.update(xd[:, :, t * sp.stride:(t + 1) * sp.stride].contiguous())
        dc.forward()
        pred = dc.noise().cpu().numpy()[0, 0]
        running = dc.cleaned(gw.GW_RUNNING).cpu().numpy()[0, 0]
        rms[t] = float(np.sqrt(np.mean(pred.astype(np.float64) ** 2)))
        got[("pred", t)] = pred
        got[("cleaned_running", t)] = running
    checked = 0
    for k, t, i, v in recs:
        if (k, t) in got:
            assert abs(float(got[(k, t)][i]) - v) <= util.ELEM_RMS * rms[t], (k, t, i, float(got[(k, t)][i]), v)
            checked += 1
    assert checked >= 40


# ------------------------------------------------------- C1 and C3 at full size, long streams
@pytest.mark.gpu
def test_c1_full_rate_streaming_bf16_steady_state():
    """BASELINE.json configs[1]: one stream, 21 witnesses, W = 32768, S = 1024 (k = 32), bf16, 40 updates: the first
    updates (warm-up, partly-zero windows) and the 8 steady-state updates after all 32 overlapping windows exist."""
    cfg = S.config_c1()
    sp = cfg.stream
    dtype = gw.GW_BF16
    dc_params, _ = util.make_params(cfg)
    n_up = 40
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, None, dtype)
    orc = util.make_stream_oracle(cfg, dc_params, None, dtype, n_up)
    xd = _dev(x)
    et = util.elem_tol(dtype)
    worst = worst_l2 = 0.0
    for t in range(n_up):
        stream.update(xd[:, :, t * sp.stride:(t + 1) * sp.stride].contiguous())
        dc.forward()
        pred = dc.noise().cpu().numpy()[0, 0]
        final = dc.cleaned(gw.GW_FINAL).cpu().numpy()[0, 0]
        ref = orc.update(x[0][:, t * sp.stride:(t + 1) * sp.stride])
        if t < 3 or t >= 31:
            r = util.check_network_output(pred, ref["pred"][0], f"C1 pred update {t}", elem=et)
            util.check_network_output(final, ref["cleaned_final"][0], f"C1 final update {t}", rms_ref=ref["pred"][0], elem=et)
            worst = max(worst, r[1]); worst_l2 = max(worst_l2, r[0])
    # reported, not asserted: north_star's per-element bar (2e-2 RMS) against the UNROUNDED-activation fp64 oracle is out
    # of reach of any bf16-storage implementation (tests/test_oracle_pins.py::test_bf16_activation_storage_alone_...)
    print(f"C1 bf16 vs fp64 oracle: worst |d|/RMS {worst:.3e} ({'meets' if worst <= util.ELEM_RMS else 'MISSES'} north_star's "
          f"2e-2; asserted bar {et}), worst rel L2 {worst_l2:.3e} (bar {util.REL_L2})")


@pytest.mark.gpu
def test_c3_ten_minute_stream_first_and_late_blocks():
    """BASELINE.json configs[3]: 2 detectors x 21 witnesses, W = 32768, S = 512 (k = 64), classifier on the last
    second, 4800 updates = 10 min, through the CUDA graph.  Full chain (raw prediction, final cleaned samples, score)
    against the oracle on the first 72 updates and on the last 72; the oracle skips the updates in between (its
    overlap-add state is rebuilt over the 63 updates before the late block, which are computed but not compared)."""
    cfg = S.config_c3(1)
    sp = cfg.stream
    dtype = gw.GW_FP16
    k = sp.window // sp.stride
    n_up, blk = 4800, 72
    dc_params, bbh_params = util.make_params(cfg)
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype)
    # [update][stream][channel][S], resident before the loop: every step's input is a contiguous view, no copies race
    xc = torch.from_numpy(np.ascontiguousarray(x.reshape(1, sp.channels, n_up, sp.stride).transpose(2, 0, 1, 3))).cuda()
    cs = torch.cuda.Stream()
    scores_d = torch.zeros(1, device="cuda")
    final_d = torch.zeros((1, sp.n_det, sp.stride), device="cuda")
    torch.cuda.synchronize()
    keep = {}
    for t in range(n_up):
        pipe.step(xc[t], scores_d, final_d, cs)
        if t < blk or t >= n_up - blk:
            cs.synchronize()
            keep[t] = (dc.noise().cpu().numpy()[0], final_d.cpu().numpy()[0].copy(), float(scores_d.cpu()[0]))
    cs.synchronize()
    orc = util.make_stream_oracle(cfg, dc_params, bbh_params, dtype, n_up)
    first_late = n_up - blk - (k - 1)
    for t in range(n_up):
        new = x[0][:, t * sp.stride:(t + 1) * sp.stride]
        if blk <= t < first_late:
            orc.skip(new)
            continue
        ref = orc.update(new)
        if t in keep:
            pred, final, score = keep[t]
            for d in range(sp.n_det):
                util.check_network_output(pred[d], ref["pred"][d], f"C3 pred update {t} det {d}")
                util.check_network_output(final[d], ref["cleaned_final"][d], f"C3 final update {t} det {d}", rms_ref=ref["pred"][d])
            assert abs(score - ref["score"]) <= util.SCORE_ABS, (t, score, ref["score"])


@pytest.mark.gpu
def test_step_profile_decomposes_the_graph_step_and_outputs_rotate_without_recapture():
    """gwstream_diag.h: gw_step_profile stamps every kernel INSIDE the replayed graph; the exclusive shares add up to
    the device span of the step, and the profiled step computes the same numbers as a plain gw_step.  Also the
    ADVICE item: new output buffers are node-parameter updates (results land in the buffer passed to THAT call)."""
    cfg = S.config_small_ensemble(3)
    sp = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    n_up = 8
    x = synth.multi_stream(cfg.seed, sp, n_up * sp.stride)
    xc = torch.from_numpy(np.ascontiguousarray(x.reshape(sp.n_streams, sp.channels, n_up, sp.stride).transpose(2, 0, 1, 3))).cuda()
    res = {}
    for mode in ("plain", "profiled"):
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, gw.GW_FP16)
        cs = torch.cuda.Stream()
        scs = [torch.zeros(sp.n_streams, device="cuda") for _ in range(3)]
        fins = [torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda") for _ in range(3)]
        torch.cuda.synchronize()
        out = []
        for t in range(n_up):
            b = t % 3                                    # rotate output buffers every step
            if mode == "profiled" and t >= 2:
                rows = pipe.step_profile(xc[t], scs[b], fins[b], cs)
                labels = [r["label"] for r in rows]
                assert labels[0] == "snapshot_append" and "aggregate" in labels and labels[-1] == "bbh_fused"
                assert len(rows) == pipe.graph_nodes() == 9            # append, 6 DeepClean kernels (layers 0 + 1 and the tail fused), overlap-add, classifier
                prev_end, span = 0.0, 0.0
                for r in rows:
                    assert r["end_us"] > r["begin_us"] >= 0.0, r
                    assert 300.0 < r["sm_mhz"] < 2500.0, r       # clock64 / %globaltimer of the kernel's CTA 0
                    span += max(0.0, r["end_us"] - max(r["begin_us"], prev_end))
                    prev_end = max(prev_end, r["end_us"])
                # exclusive shares + idle gaps between kernels = end of the last kernel
                assert 0.5 * prev_end < span <= prev_end + 1e-6 and prev_end < 5000.0, (span, prev_end)
                assert sum(r["flops"] for r in rows if r["label"].startswith("gemm.dc")) > 1e9
            else:
                pipe.step(xc[t], scs[b], fins[b], cs)
            cs.synchronize()
            out.append((fins[b].cpu().numpy().copy(), scs[b].cpu().numpy().copy()))
        res[mode] = out
    for t in range(n_up):
        assert np.array_equal(res["plain"][t][0], res["profiled"][t][0]), t
        assert np.array_equal(res["plain"][t][1], res["profiled"][t][1]), t
    assert any(np.any(res["plain"][t][0] != res["plain"][t + 1][0]) for t in range(n_up - 1))


@pytest.mark.gpu
def test_mma_probe_reports_the_operand_read_law():
    """gw_probe_mma_cycles: the measured cycles per tcgen05.mma follow max(N/2, 32 + N/4) within 15 % on this class of
    device (the thin layers' shared-memory roofline in DESIGN.md rests on it); bad N is rejected."""
    got = gw.probe_mma_cycles()
    for n, (issue, done) in got.items():
        law = max(n / 2, 32 + n / 4)
        assert 0.85 * law <= done <= 1.15 * law, (n, issue, done, law)
    with pytest.raises(gw.GwError):
        gw.probe_mma_cycles((48,))


@pytest.mark.gpu
def test_handles_release_their_device_memory():
    """Create / run / destroy every kind of handle a few times: free device memory returns to where it started
    (the engine owns all persistent state, include/gwstream.h)."""
    import gc
    cfg = S.config_small_ensemble(2)
    sp = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    x = _dev(synth.multi_stream(cfg.seed, sp, 2 * sp.stride))
    one = S.StreamSpec(1, sp.n_det, sp.fs, sp.window, sp.stride, sp.n_witness)
    seg = _dev(synth.stream_channels(1, one, sp.window + 3 * sp.stride))
    scores_h = torch.zeros(sp.n_streams).pin_memory()
    final_h = torch.zeros((sp.n_streams, sp.n_det, sp.stride)).pin_memory()
    xin = torch.from_numpy(np.ascontiguousarray(x[:, :, :sp.stride].cpu().numpy())).pin_memory()

    def cycle():
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, gw.GW_FP16)
        cs = torch.cuda.Stream()
        sc = torch.zeros(sp.n_streams, device="cuda")
        fin = torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda")
        cs.wait_stream(torch.cuda.current_stream())
        pipe.step(x[:, :, :sp.stride].contiguous(), sc, fin, cs)
        pipe.step_host_async(xin, scores_h, final_h, cs)
        cs.synchronize()
        off = gw.Offline(one, cfg.dc_layers, dc_params, 4, gw.GW_FP16)
        off.run(seg)
        torch.cuda.synchronize()
        for h in (pipe, bbh, dc, stream, off):
            h.__del__()
        del sc, fin

    cycle()                                              # first cycle: CUDA module load, allocator pools
    gc.collect(); torch.cuda.synchronize(); torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        cycle()
    gc.collect(); torch.cuda.synchronize(); torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 8 * 2**20, (free0, free1)


@pytest.mark.gpu
@pytest.mark.parametrize("W,S_,n,dtype", [(2048, 256, 3, gw.GW_FP16), (4096, 512, 2, gw.GW_BF16), (32768, 512, 3, gw.GW_FP16)])
def test_first_two_layers_as_one_kernel_are_bit_identical(W, S_, n, dtype):
    """gw_options.fuse_head (default): layers 0 and 1 run as one kernel -- two tiles of layer 0 become, activated and in
    shared memory, one operand tile of layer 1 (super-tiles of 125 rows overlapping by three position pairs; 17 to 66 of them
    per window here, walked backwards under the snake order).  The same products in the same order as the two kernels:
    prediction, final samples, scores and every stored activation from layer 1 on must be array_equal, and the graph has one
    kernel fewer."""
    cfg0 = S.config_c3(n, S_, W)
    cfg = S.Config("head", cfg0.stream, cfg0.dc_layers, cfg0.bbh_convs, cfg0.bbh_dense, min(4096, W // 2), 0, 31)
    sp = cfg.stream
    n_up = 6
    dc_params, bbh_params = util.make_params(cfg)
    x = synth.multi_stream(cfg.seed, sp, n_up * S_)
    xc = torch.from_numpy(np.ascontiguousarray(x.reshape(n, sp.channels, n_up, S_).transpose(2, 0, 1, 3))).cuda()
    outs, acts, nodes = {}, {}, {}
    for fuse in (1, 0):
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, opts=gw.Options(fuse_head=fuse))
        cs = torch.cuda.Stream()
        sc = torch.zeros(n, device="cuda")
        fin = torch.zeros((n, sp.n_det, S_), device="cuda")
        torch.cuda.synchronize()
        res = []
        for t in range(n_up):
            pipe.step(xc[t], sc, fin, cs)
            cs.synchronize()
            res.append((dc.noise().cpu().numpy(), fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
        outs[fuse], nodes[fuse] = res, pipe.graph_nodes()
        acts[fuse] = [dc.activation(li).cpu().view(torch.int16).numpy() for li in range(1, len(cfg.dc_layers) - 2)]
    assert nodes[1] == nodes[0] - 1, nodes
    for li, (a1, a0) in enumerate(zip(acts[1], acts[0])):
        assert np.array_equal(a1, a0), ("activation after layer", li + 1, np.argwhere(a1 != a0)[:4])
    for t in range(n_up):
        for a, b, what in zip(outs[1][t], outs[0][t], ("pred", "final", "scores")):
            assert np.array_equal(a, b), (t, what)


@pytest.mark.gpu
def test_scheduling_switches_are_bit_identical():
    """include/gwstream.h promises that gw_options.pdl / snake / two_sm / skip_zeros change scheduling (or skip exact
    zeros) only.  C3-shaped layers at full window length (the CTA-pair kernel needs an even number of 128-row tiles),
    three streams so that CTAs walk several work items; every switch off in turn, compared bitwise with all on."""
    cfg = S.config_c3(3, 512, 32768)
    sp = cfg.stream
    dc_params, bbh_params = util.make_params(cfg)
    n_up = 2
    xc = torch.from_numpy(np.ascontiguousarray(
        synth.multi_stream(cfg.seed, sp, n_up * sp.stride).reshape(sp.n_streams, sp.channels, n_up, sp.stride).transpose(2, 0, 1, 3))).cuda()
    switches = ("pdl", "snake", "two_sm", "skip_zeros")

    def run(opts=None):
        stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, gw.GW_FP16, opts=opts)
        cs = torch.cuda.Stream()
        sc = torch.zeros(sp.n_streams, device="cuda")
        fin = torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda")
        torch.cuda.synchronize()
        out = []
        for t in range(n_up):
            pipe.step(xc[t], sc, fin, cs)
            cs.synchronize()
            out.append((dc.noise().cpu().numpy(), fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
        return out

    base = run()
    for name in switches:
        got = run(gw.Options(**{name: 0}))
        for t in range(n_up):
            for a, b, what in zip(got[t], base[t], ("pred", "final", "scores")):
                assert np.array_equal(a, b), (name, t, what)


@pytest.mark.gpu
def test_random_shapes_and_option_combinations_are_bit_identical():
    """Seeded draws of (window, stride, streams, dtype) and of every gw_options switch at once, against the plain path
    (nothing fused, full recompute, no PDL / snake / CTA pairs / zero skipping) with the same fuse_tail -- the one switch
    the header states as 'within rounding'.  Prediction and final samples array_equal on warm-up and steady-state updates;
    scores array_equal with the three-kernel classifier, within the score bar with the one-kernel one (other arithmetic)."""
    import random
    rng = random.Random(20260)
    cases = 0
    for _ in range(10):
        W = rng.choice([2048, 4096, 6144, 8192, 16384])
        S_ = rng.choice([s for s in (16, 64, 128, 256, 512, 1024, 2048) if s <= W // 2 and W % s == 0])
        n = rng.choice([1, 2, 3, 4, 5, 8])
        dtype = rng.choice([gw.GW_FP16, gw.GW_BF16])
        cfg0 = S.config_c3(n, S_, W)
        cfg = S.Config("mix", cfg0.stream, cfg0.dc_layers, cfg0.bbh_convs, cfg0.bbh_dense, 512 * max(1, min(4096, W // 2) // 512), 0,
                       rng.randrange(1000))
        sp = cfg.stream
        n_up = min(W // S_ + 4, 24)
        dc_params, bbh_params = util.make_params(cfg)
        xc = torch.from_numpy(np.ascontiguousarray(
            synth.multi_stream(cfg.seed, sp, n_up * S_).reshape(n, sp.channels, n_up, S_).transpose(2, 0, 1, 3))).cuda()

        def run(opts):
            stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype, opts=opts)
            cs = torch.cuda.Stream()
            sc = torch.zeros(n, device="cuda")
            fin = torch.zeros((n, sp.n_det, S_), device="cuda")
            torch.cuda.synchronize()
            out = []
            for t in range(n_up):
                pipe.step(xc[t], sc, fin, cs)
                cs.synchronize()
                if t < 2 or t % 4 == 0 or t >= n_up - 2:
                    out.append((dc.noise().cpu().numpy(), fin.cpu().numpy().copy(), sc.cpu().numpy().copy()))
            return out

        plain = {ft: run(gw.Options(fuse_tail=ft, fuse_head=0, fuse_bbh=0, incremental=0, snake=0, pdl=0, two_sm=0, skip_zeros=0))
                 for ft in (0, 1)}
        for trial in range(3):
            o = {name: rng.randint(0, 1) for name in ("fuse_tail", "fuse_head", "fuse_bbh", "incremental", "snake", "pdl", "two_sm", "skip_zeros")}
            if trial == 0:
                o = dict(fuse_tail=1, fuse_head=1, fuse_bbh=1, incremental=1, snake=1, pdl=1, two_sm=1, skip_zeros=1)
            if o["incremental"] and (W % 2048 or S_ % 16 or not o["fuse_tail"]):
                o["incremental"] = 0                     # shapes / combinations the incremental path refuses (tested elsewhere)
            got = run(gw.Options(**o))
            cases += 1
            for (p0, f0, s0), (p1, f1, s1) in zip(plain[o["fuse_tail"]], got):
                assert np.array_equal(p0, p1), ("pred", W, S_, n, dtype, o)
                assert np.array_equal(f0, f1), ("final", W, S_, n, dtype, o)
                if o["fuse_bbh"]:
                    assert np.abs(s0 - s1).max() <= 5e-3, ("scores", W, S_, n, dtype, o)
                else:
                    assert np.array_equal(s0, s1), ("scores", W, S_, n, dtype, o)
    assert cases == 30


@pytest.mark.gpu
def test_mufu_probe_reports_sixteen_results_per_clock_per_sm():
    """gw_probe_mufu_rate: tanh.approx.f32 retires 16 per clock per SM once the SM holds >= 256 threads, the packed f16x2
    form gives the same 16 RESULTS per clock (two operations per instruction), the bf16 engine's ex2 + rcp form 8 tanh per
    clock: the MUFU floor under the thin layers (bench.py's mufu_frac) rests on these."""
    for threads in (256, 512):
        r = gw.probe_mufu_rate(0, threads)
        assert 15.0 <= r <= 16.2, (threads, r)
    assert 15.0 <= gw.probe_mufu_rate(1, 512) <= 16.2
    assert 7.5 <= gw.probe_mufu_rate(2, 512) <= 8.1
    with pytest.raises(gw.GwError):
        gw.probe_mufu_rate(3, 512)
    with pytest.raises(gw.GwError):
        gw.probe_mufu_rate(0, 100)
