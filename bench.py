#!/usr/bin/env python
"""bench.py -- data-seconds/s of the end-to-end ensemble (snapshotter -> 2x DeepClean -> Hann
overlap-add + subtraction -> BBH classifier) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl native|reference]
                    [--streams n] [--stride S] [--dtype fp16|bf16]

A "step" is one update of ALL n streams (BASELINE.json configs[4]: independent config-3 ensemble
streams batched into one CUDA-graph launch per stride): n*S/fs data-seconds.  Inputs are seeded
synthetic data shaped like the paper's workload, resident in HBM for
`value`, in pinned host memory for `e2e`.  N > 1 (torchrun): every rank runs its own n streams, no
collective on the data path (streams are independent), value = sum over ranks
/ max time: "scaling": "weak".

--impl reference times the CPU oracle (oracle/, fp64 direct loops) as it stands on the host cores,
each step being ONE stream's update (a bounded sample of the same workload).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2108_12430_b200 import shard               # noqa: E402
from paper_2108_12430_b200 import specs as S          # noqa: E402
from paper_2108_12430_b200 import synth               # noqa: E402

METRIC = "data-seconds/s processed (DeepClean+BBH)"
UNIT = "data-seconds/s"
FS = 4096
WINDOW = 32768
SEG_SECONDS = 16          # looped device-resident input segment per stream (BASELINE.json configs[4])
SWEEP_STREAMS = (1, 16, 128, 512)      # BASELINE.json configs[4]
SWEEP_STRIDES = (256, 512, 1024)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def make_params(cfg):
    dc = [synth.deepclean_params(cfg.seed * 100 + d, cfg.dc_layers) for d in range(cfg.stream.n_det)]
    bbh = synth.bbh_params(cfg.seed * 100 + 50, cfg.bbh_convs, cfg.bbh_dense)
    return dc, bbh


def make_input_chunks(cfg, n_chunks: int) -> np.ndarray:
    """[n_chunks][n][C][S] float32: chunk k holds update k's strictly new samples for every stream.
    Four streams are synthesised from the recipe; the rest are time-rolled copies (values do not
    affect timing: the path has no data-dependent control flow)."""
    sp = cfg.stream
    T = n_chunks * sp.stride
    base = [synth.stream_channels(cfg.seed + i, sp, T) for i in range(min(4, sp.n_streams))]
    out = np.empty((n_chunks, sp.n_streams, sp.channels, sp.stride), dtype=np.float32)
    for i in range(sp.n_streams):
        x = np.roll(base[i % len(base)], 977 * (i // len(base)), axis=1)
        out[:, i] = x.reshape(sp.channels, n_chunks, sp.stride).transpose(1, 0, 2)
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"tensor_tflops": float(p.get("bf16_tflops_sustained", p.get("bf16_tflops", 1590.0))),
                "tensor_tflops_burst": float(p.get("bf16_tflops", 1590.0)), "hbm_gbs": float(p.get("hbm_gbs", 6650.0)),
                "source": "measured (MEASURED_PEAKS.json; sustained bf16 GEMM, fp16 shares the pipe rate)"}
    return {"tensor_tflops": 1400.0, "tensor_tflops_burst": 1590.0, "hbm_gbs": 6650.0,
            "source": "fallback (B200_PROFILING.md)"}


# ------------------------------------------------------------------------------- CPU oracle leg
def oracle_rate(cfg, dtype_name: str, n_updates: int, budget_s: float = 1e9):
    """Time the oracle (as it stands) on up to `n_updates` updates of ONE stream of the same workload;
    stops early once `budget_s` seconds of oracle time are spent (the run must end within minutes)."""
    import oracle
    od = oracle.DT_BF16 if dtype_name == "bf16" else oracle.DT_FP16
    sp = cfg.stream
    one = S.StreamSpec(1, sp.n_det, sp.fs, sp.window, sp.stride, sp.n_witness)
    dc_params, (cp, dp) = make_params(cfg)
    rows = [(one.witness_rows(d), one.strain_row(d)) for d in range(one.n_det)]
    dc = [(cfg.dc_layers, [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.dc_layers, dc_params[d])])
          for d in range(one.n_det)]
    bbh = (cfg.bbh_convs, [oracle.prepare_conv(l, p, od) for l, p in zip(cfg.bbh_convs, cp)],
           [oracle.prepare_dense(p) for p in dp], cfg.bbh_len)
    so = oracle.StreamOracle(one.channels, one.window, one.stride, rows, dc, bbh, max_updates=n_updates + 1)
    x = synth.stream_channels(cfg.seed, one, (n_updates + 1) * one.stride)
    times = []
    for t in range(n_updates):
        t0 = time.perf_counter()
        so.update(x[:, t * one.stride:(t + 1) * one.stride])
        times.append(time.perf_counter() - t0)
        if sum(times) > budget_s:
            break
    return times, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = S.config_c3(args.streams, args.stride, WINDOW)
    if int(os.environ.get("WORLD_SIZE", "1")) > 1 and os.environ.get("OMP_NUM_THREADS") == "1":
        # torchrun pins every rank to one OpenMP thread; the other ranks do no work here, so rank 0 takes the host's cores
        # as in the N = 1 run (the line's `cores` says what was used)
        import oracle
        oracle.set_num_threads(len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    times, cores = oracle_rate(cfg, args.dtype, args.warmup + args.steps, budget_s=args.reference_budget)
    timed = times[args.warmup:] if len(times) > args.warmup else times[-1:]
    sec = sum(timed)
    ds = args.stride / FS
    value = len(timed) * ds / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(timed), "steps_requested": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / len(timed),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"C3 ensemble, ONE stream per step (bounded sample of C4 n={args.streams}), "
                               f"W={WINDOW}, S={args.stride}, fs={FS}", "weights_rounded_to": args.dtype},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{len(timed)} updates of one 2-detector stream"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------ native leg
NOMINAL_TFLOPS = 2250.0       # B200 dense bf16/fp16 spec-sheet figure (B200_PROFILING.md, "nominal, for context")
NOMINAL_HBM_GBS = 7700.0


class Engine:
    """One engine instance (n streams of the C3 ensemble) plus the measurement legs bench.py runs on it."""

    def __init__(self, gw, torch, args, n_streams, stride, dtype, opts, chunks_h=None, seg_seconds=None, local=0):
        self.gw, self.torch, self.args = gw, torch, args
        self.cfg = S.config_c3(n_streams, stride, WINDOW)
        self.sp = self.cfg.stream
        self.dtype_name = dtype
        self.n_chunks = (seg_seconds or args.seg_seconds) * FS // stride
        self.dc_params, self.bbh_params = make_params(self.cfg)
        if chunks_h is None:
            t0 = time.time()
            chunks_h = torch.from_numpy(make_input_chunks(self.cfg, self.n_chunks)).pin_memory()
            log(f"inputs {tuple(chunks_h.shape)} ({chunks_h.numel() * 4 / 2**20:.0f} MiB) in {time.time() - t0:.1f}s")
        self.chunks_h = chunks_h
        self.chunks_d = chunks_h.cuda()
        self.stream, self.dc, self.bbh, self.pipe = gw.build_ensemble(
            self.cfg, self.dc_params, self.bbh_params, gw.GW_BF16 if dtype == "bf16" else gw.GW_FP16, opts=opts)
        self.cs = torch.cuda.Stream()
        self.scores = torch.zeros(self.sp.n_streams, device="cuda")
        self.final = torch.zeros((self.sp.n_streams, self.sp.n_det, self.sp.stride), device="cuda")
        self.step_no = 0
        self.ds_per_step = self.sp.n_streams * self.sp.stride / FS

    def step(self):
        self.pipe.step(self.chunks_d[self.step_no % self.n_chunks], self.scores, self.final, self.cs)
        self.step_no += 1

    def timed(self, k):
        """k back-to-back graph steps between two CUDA events on the launch stream -> total ms."""
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.cs)
        for _ in range(k):
            self.step()
        e1.record(self.cs)
        self.cs.synchronize()
        return e0.elapsed_time(e1)

    def latency(self, n):
        lat = []
        for _ in range(n):
            t0 = time.perf_counter()
            self.step()
            self.cs.synchronize()
            lat.append((time.perf_counter() - t0) * 1e3)
        lat.sort()
        return {"p50_ms": lat[len(lat) // 2], "p99_ms": lat[min(len(lat) - 1, int(len(lat) * 0.99))],
                "samples": len(lat), "per_stream_p50_ms": lat[len(lat) // 2] / self.sp.n_streams,
                "realtime_budget_ms": 1e3 * self.sp.stride / FS,
                "what": "host clock, gw_step launch -> stream synchronize, whole batch of n streams"}

    def e2e(self, k, world=1):
        """End to end through the C ABI with HOST buffers (pinned): H2D of every step's samples and D2H of its scores
        and final cleaned samples inside the timed region.  The outputs ROTATE over four buffer pairs (a consumer reads
        step i while step i+1 runs; different output pointers are node-parameter updates of the graph, never a
        re-capture) and every step's results are read on the host (summed) inside the timed region, one step behind."""
        torch, sp = self.torch, self.sp
        nbuf = 4
        sc_h = [torch.zeros(sp.n_streams).pin_memory() for _ in range(nbuf)]
        fin_h = [torch.zeros((sp.n_streams, sp.n_det, sp.stride)).pin_memory() for _ in range(nbuf)]
        evs = [torch.cuda.Event() for _ in range(nbuf)]
        for i in range(nbuf):                         # warm-up: capture + every buffer pair seen once
            self.pipe.step_host_async(self.chunks_h[self.step_no % self.n_chunks], sc_h[i], fin_h[i], self.cs)
            self.step_no += 1
        torch.cuda.synchronize()
        checksum = 0.0
        t0 = time.perf_counter()
        for i in range(k):
            b = i % nbuf
            self.pipe.step_host_async(self.chunks_h[self.step_no % self.n_chunks], sc_h[b], fin_h[b], self.cs)
            evs[b].record(self.cs)
            self.step_no += 1
            if i >= 1:                                # consume the previous step's results while this one runs
                pb = (i - 1) % nbuf
                evs[pb].synchronize()
                checksum += float(sc_h[pb].sum()) + float(fin_h[pb].sum())
        evs[(k - 1) % nbuf].synchronize()
        checksum += float(sc_h[(k - 1) % nbuf].sum())
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        t1 = time.perf_counter()
        n_sync = min(k, 50)
        for _ in range(n_sync):                       # online regime: gw_step_host returns with the results
            self.pipe.step_host(self.chunks_h[self.step_no % self.n_chunks], sc_h[0], fin_h[0], self.cs)
            self.step_no += 1
        sync_ms = 1e3 * (time.perf_counter() - t1) / n_sync
        sec = shard.max_over_ranks(sec, device="cuda")
        return {"value": world * k * self.ds_per_step / sec, "unit": UNIT,
                "h2d_bytes_per_step": sp.n_streams * sp.channels * sp.stride * 4,
                "d2h_bytes_per_step": sp.n_streams * 4 + sp.n_streams * sp.n_det * sp.stride * 4,
                "ms_per_step": 1e3 * sec / k, "ms_per_step_synchronous": sync_ms, "output_buffers": nbuf,
                "checksum_finite": bool(np.isfinite(checksum)),
                "what": "gw_step_host_async: pinned host buffers, H2D of every step's samples and D2H of its scores and final "
                        "cleaned samples inside the timed region, outputs rotating over 4 buffer pairs and read on the host "
                        "one step behind, host clock; ms_per_step_synchronous = gw_step_host (returns with each update's results)"}

    def profile(self, reps=8, prewarm_s=0.5, ms_per_step=1.0):
        """Per-kernel device spans INSIDE the graph replay (%globaltimer stamps, gwstream_diag.h): mean over `reps`
        profiled steps of each kernel's duration and of its exclusive share excl_i = end_i - max(begin_i, end_{i-1});
        sum(excl) = device span of the step, which cannot exceed the step time measured around the launch.  The
        profiled steps follow `prewarm_s` seconds of back-to-back steps without a gap, so they run in the same clock /
        power regime as the sustained leg (the caller samples the clocks around this call)."""
        acc = {}
        order = []
        self.pipe.step_profile(self.chunks_d[self.step_no % self.n_chunks], self.scores, self.final, self.cs)   # capture
        self.step_no += 1
        for _ in range(int(prewarm_s * 1e3 / max(ms_per_step, 1e-3))):
            self.step()
        for it in range(reps + 1):
            rows = self.pipe.step_profile(self.chunks_d[self.step_no % self.n_chunks], self.scores, self.final, self.cs)
            self.step_no += 1
            if it == 0:
                continue
            prev_end = 0.0
            for r in rows:
                a = acc.setdefault(r["label"], {"us": 0.0, "excl_us": 0.0, "flops": 0.0, "smem_bytes": 0.0, "sm_mhz": 0.0})
                a["sm_mhz"] += r.get("sm_mhz", 0.0) / reps
                if r["label"] not in order:
                    order.append(r["label"])
                a["us"] += (r["end_us"] - r["begin_us"]) / reps
                a["excl_us"] += max(0.0, r["end_us"] - max(r["begin_us"], prev_end)) / reps
                a["flops"], a["smem_bytes"] = r["flops"], r["smem_bytes"]
                prev_end = max(prev_end, r["end_us"])
        return order, acc

    def close(self):
        for h in (self.pipe, self.bbh, self.dc, self.stream):
            h.close()
        del self.chunks_d


def kernel_table(eng, order, acc, pk, sm_mhz, sms, full=True):
    """Per-kernel dict for the bench line: duration and exclusive share (us, from the graph-replay stamps), TFLOP/s on
    the exclusive time for the conv GEMMs (executed algorithmic FLOPs), GB/s for the bandwidth kernels."""
    sp, cfg = eng.sp, eng.cfg
    nd, nw = sp.n_det, sp.n_witness
    # ALGORITHMIC bytes per launch
    hbm_bytes = {
        "append": sp.n_streams * sp.channels * sp.stride * 8,                       # read new + write ring
        "ring16_append": sp.n_streams * nd * sp.stride * (nw * 4 + 2 * 32 * 2),     # read fp32, write both mirror copies
        "snapshot_append": sp.n_streams * (sp.channels * sp.stride * 8 + nd * sp.stride * 2 * 32 * 2),  # a1 + a2 fused
        # a5 as launched inside the step: reads p_t and acc (8 W - 4 S: the newest stride's accumulators start from zero),
        # writes acc (4 W); the strain is read only where a cleaned sample leaves the kernel -- the S final samples and the
        # L_b classifier samples (8 (S + L_b) read + written); the running cleaned window is NOT written on this path
        "aggregate": sp.n_streams * nd * (sp.window * 12 + sp.stride * 4 + cfg.bbh_len * 8),
        "bbh_conv1": sp.n_streams * (nd * cfg.bbh_len * 4 + (cfg.bbh_len // 4) * 32 * 2),
        "bbh_fused": sp.n_streams * (nd * cfg.bbh_len * 4 + 4),                      # the window in, one score out
    }
    smem_peak_gbs = sms * 128 * sm_mhz * 1e6 / 1e9
    # MUFU operations of a whole-window DeepClean launch: one per tanh (fp16: tanh.approx.f32) or two (bf16: ex2 + rcp); the
    # pipe retires 16 per clock per SM (measured: 15.99 with 512-1024 threads per SM, any operand width -- f16x2 / bf16x2 are
    # two operations).  Zone launches (incremental path) are not counted: their rows are a fraction of the layer.
    mufu_ops = {}
    if full:
        per_tanh = 2 if eng.dtype_name == "bf16" else 1
        lens, tanh = [sp.window], []
        for l in cfg.dc_layers:
            lens.append(l.lout(lens[-1]))
            tanh.append(sp.n_streams * nd * lens[-1] * l.cout * per_tanh if l.act == S.ACT_TANH else 0)
        for k in order:
            if k.startswith("gemm.dc"):
                mufu_ops[k] = sum(tanh[int(i)] for i in k[len("gemm.dc"):].split("+"))   # the fused tail's last layer is linear
    out = {}
    for k in order:
        a = acc[k]
        row = {"us": round(a["us"], 2), "excl_us": round(a["excl_us"], 2), "sm_mhz": round(a["sm_mhz"])}
        t = a["excl_us"] * 1e-6
        mhz = a["sm_mhz"] or sm_mhz                    # the clock THIS kernel ran at (clock64 / %globaltimer of its CTA 0)
        if a["flops"] and t > 0:
            row["tflops"] = round(a["flops"] / t / 1e12, 1)
            row["tflops_own_span"] = round(a["flops"] / (a["us"] * 1e-6) / 1e12, 1)
            # against what the tensor cores can do AT THAT CLOCK: 8192 dense 16-bit FLOP per clock per SM (2.25 PFLOP/s
            # nominal = 148 SMs x 8192 x 1.855 GHz)
            row["frac_of_tensor_peak_at_clock"] = round(a["flops"] / t / (sms * 8192.0 * mhz * 1e6), 3)
        if a["smem_bytes"] and a["us"] > 0:
            gbs = a["smem_bytes"] / (a["us"] * 1e-6) / 1e9
            row.update({"smem_gbs": round(gbs, 1), "smem_frac": round(gbs / (sms * 128 * mhz * 1e6 / 1e9), 3)})
        if mufu_ops.get(k) and a["us"] > 0:
            row.update({"mufu_ops": mufu_ops[k], "mufu_frac": round(mufu_ops[k] / (a["us"] * 1e-6) / (sms * 16.0 * mhz * 1e6), 3)})
        if k in hbm_bytes and a["us"] > 0:
            gbs = hbm_bytes[k] / (a["us"] * 1e-6) / 1e9
            row.update({"gbs": round(gbs, 1), "hbm_frac": round(gbs / pk["hbm_gbs"], 3),
                        "hbm_frac_nominal": round(gbs / NOMINAL_HBM_GBS, 3)})
        out[k] = row
    return out, smem_peak_gbs


def run_native(args):
    import torch
    import torch.distributed as dist
    from paper_2108_12430_b200 import binding as gw

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    opts = gw.Options(pdl=not args.no_pdl, snake=not args.no_snake, skip_zeros=not args.no_skip, two_sm=not args.no_2sm,
                      incremental=args.incremental)
    eng = Engine(gw, torch, args, args.streams, args.stride, args.dtype, opts, local=local)
    sp, cfg = eng.sp, eng.cfg

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    W_, K = max(args.warmup, 3), args.steps
    for _ in range(W_):
        eng.step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = gw.kernel_launches()
    ms_total = eng.timed(K)
    barrier()
    launches = gw.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms_total = shard.max_over_ranks(ms_total, device="cuda")
    value = world * K * eng.ds_per_step / (ms_total / 1e3)

    if args.timed_only:
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
                              "warmup": W_, "ms_per_step": ms_total / K, "gpu_launches": int(launches),
                              "note": "--timed-only run (profiling aid), not a bench line"}), flush=True)
        return

    # sustained regime: back-to-back steps for >= args.sustained_seconds with the clock sampler running during it
    sustained = None
    if args.sustained_seconds > 0:
        n_sus = max(K, int(args.sustained_seconds * 1e3 / (ms_total / K)) + 1)
        s2 = ClockSampler(local)
        if rank == 0:
            s2.start()
        ms_sus = shard.max_over_ranks(eng.timed(n_sus), device="cuda")
        c2 = s2.stop() if rank == 0 else None
        sustained = {"value": world * n_sus * eng.ds_per_step / (ms_sus / 1e3), "unit": UNIT, "steps": n_sus,
                     "seconds": ms_sus / 1e3, "ms_per_step": ms_sus / n_sus, "clocks": c2}

    latency = eng.latency(min(max(K, 50), 5000))
    e2e = eng.e2e(K, world)

    # ---- roofline of the dominant kernel family (all conv-GEMM launches of a step), regime-honest
    s5 = ClockSampler(local)
    if rank == 0:
        s5.start()
    order, acc = eng.profile(ms_per_step=ms_total / K)
    clocks_profile = s5.stop() if rank == 0 else None
    graph_nodes = eng.pipe.graph_nodes()
    pk = peaks()
    sm_mhz_sus = (clocks_profile or {}).get("sm_mhz") or ((sustained or {}).get("clocks") or {}).get("sm_mhz") or 1700.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    kernels, smem_peak_gbs = kernel_table(eng, order, acc, pk, sm_mhz_sus, sms)
    mufu_total = sum(r.get("mufu_ops", 0) for r in kernels.values())
    mufu = {"unit": "MUFU operations (tanh of the DeepClean epilogues)", "ops_per_step": mufu_total, "peak_per_clock_per_sm": 16,
            "us_at_the_profiled_clock": round(mufu_total / (sms * 16.0 * sm_mhz_sus), 1),
            "what": "time the step's tanh evaluations occupy the MUFU pipe of every SM at the profiled steps' clock: a second floor "
                    "under the conv kernels beside the tensor pipe (per kernel: kernels[..].mufu_frac)"}
    gemm_us = sum(a["excl_us"] for k, a in acc.items() if k.startswith("gemm."))
    gemm_fl = sum(a["flops"] for k, a in acc.items() if k.startswith("gemm."))
    span_us = sum(a["excl_us"] for a in acc.values())
    achieved = gemm_fl / (gemm_us * 1e-6) / 1e12 if gemm_us > 0 else 0.0
    # which regime were the per-kernel times taken in?  The profiled steps are a handful of launches after idle gaps
    # (boost clocks) when the whole run is short; a run that just spent seconds back to back sits at the power cap.
    burst = False                                  # the profiled steps directly follow 0.5 s of back-to-back steps
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get("conv_gemm_dram_bytes_per_launch")
    # the same family over the SUSTAINED step: its share of the step (from the stamps) x the sustained step time
    sus_ms = sustained["ms_per_step"] if sustained else ms_total / K
    gemm_share = gemm_us / span_us if span_us else None
    achieved_sus = gemm_fl / (gemm_share * sus_ms * 1e-3) / 1e12 if gemm_share else 0.0
    peak = pk["tensor_tflops_burst"] if burst else pk["tensor_tflops"]
    roofline = {"bound": "tensor", "kernel": "k_conv_gemm_umma + k_conv_gemm_2sm (all conv-GEMM launches of one step)",
                "achieved": achieved_sus, "peak": peak, "unit": "TFLOP/s", "frac": achieved_sus / peak,
                "regime": "burst" if burst else "sustained", "clocks_profiled_steps": clocks_profile,
                "frac_burst": achieved / pk["tensor_tflops_burst"], "frac_sustained": achieved_sus / pk["tensor_tflops"],
                "frac_nominal": achieved_sus / NOMINAL_TFLOPS,
                "achieved_profiled_steps": achieved, "traffic": traffic, "peak_source": pk["source"],
                "peaks": {"burst_tflops": pk["tensor_tflops_burst"], "sustained_tflops": pk["tensor_tflops"], "nominal_tflops": NOMINAL_TFLOPS},
                "flops_per_step": gemm_fl, "us_per_step_in_kernel": gemm_us, "device_span_us": span_us,
                "share_of_step": gemm_share,
                "timing": "%globaltimer stamps written by every kernel's first / last CTA INSIDE the replay of the step's CUDA "
                          "graph (gw_step_profile); us_per_step_in_kernel = sum of the conv GEMMs' exclusive shares, device_span_us = "
                          "sum over all kernels <= ms_per_step; `achieved` = executed algorithmic FLOPs / (that share x the "
                          "sustained step time); achieved_profiled_steps = the same FLOPs / the stamped time of the profiled steps "
                          "themselves (they directly follow 0.5 s of back-to-back steps; clocks_profiled_steps), frac_burst = that "
                          "against the burst peak"}

    # ---- the exact incremental path (gw_options.incremental, D13) on the same workload
    incremental = None
    if not args.no_incremental and not args.incremental:
        eng.close()
        torch.cuda.empty_cache()
        ie = Engine(gw, torch, args, args.streams, args.stride, args.dtype,
                    gw.Options(pdl=not args.no_pdl, snake=not args.no_snake, skip_zeros=not args.no_skip, incremental=1),
                    chunks_h=eng.chunks_h, local=local)
        for _ in range(W_ + 2):
            ie.step()
        torch.cuda.synchronize()
        n_i = max(K, int(1.0e3 / 0.25))              # about a second of back-to-back steps
        s3 = ClockSampler(local)
        if rank == 0:
            s3.start()
        ms_i = shard.max_over_ranks(ie.timed(n_i), device="cuda")
        c3 = s3.stop() if rank == 0 else None
        lat_i = ie.latency(min(max(K, 50), 2000))
        e2e_i = ie.e2e(K, world)
        order_i, acc_i = ie.profile(ms_per_step=ms_i / n_i)
        kern_i, _ = kernel_table(ie, order_i, acc_i, pk, (c3 or {}).get("sm_mhz") or 1700.0, sms, full=False)
        fl_i = sum(a["flops"] for k, a in acc_i.items() if k.startswith("gemm."))
        us_i = sum(a["excl_us"] for k, a in acc_i.items() if k.startswith("gemm."))
        incremental = {"value": world * n_i * ie.ds_per_step / (ms_i / 1e3), "unit": UNIT, "steps": n_i,
                       "ms_per_step": ms_i / n_i, "latency": lat_i, "e2e": e2e_i, "clocks": c3,
                       "graph_nodes": ie.pipe.graph_nodes(),
                       "flops_executed_per_step": fl_i, "flops_full_recompute_per_step": gemm_fl,
                       "conv_work_ratio": gemm_fl / fl_i if fl_i else None,
                       "conv_tflops_on_executed_work": fl_i / (us_i * 1e-6) / 1e12 if us_i else None,
                       "device_span_us": sum(a["excl_us"] for a in acc_i.values()), "kernels": kern_i,
                       "what": "gw_options.incremental = 1: every layer's activations live in rings over absolute position and an "
                               "update recomputes only the rows near the two window edges; results are bit-identical to full "
                               "recomputation (tests/test_gpu_parity.py::test_incremental_path_is_bit_identical_to_full_recompute). "
                               "`value` above stays the full-recompute number."}
        ie.close()
        del ie
        torch.cuda.empty_cache()
        eng = None

    # ---- largest single-GPU point of configs[4]: n = 512 streams, S = 1024
    largest = None
    if not args.no_largest and world == 1:
        if eng is not None:
            eng.close(); eng = None
        torch.cuda.empty_cache()
        try:
            le = Engine(gw, torch, args, 512, 1024, args.dtype, gw.Options(), seg_seconds=1, local=local)
            for _ in range(3):
                le.step()
            torch.cuda.synchronize()
            n_l = 60
            s4 = ClockSampler(local); s4.start()
            ms_l = le.timed(n_l)
            c4 = s4.stop()
            lat_l = le.latency(30)
            largest = {"workload": "configs[4] largest point: n=512 streams, S=1024, W=32768, " + args.dtype,
                       "value": n_l * le.ds_per_step / (ms_l / 1e3), "unit": UNIT, "steps": n_l, "ms_per_step": ms_l / n_l,
                       "latency": lat_l, "clocks": c4,
                       "conv_tflops": gemm_fl * 4 / (ms_l / n_l * 1e-3) / 1e12,
                       "frac_sustained": gemm_fl * 4 / (ms_l / n_l * 1e-3) / 1e12 / pk["tensor_tflops"],
                       "frac_nominal": gemm_fl * 4 / (ms_l / n_l * 1e-3) / 1e12 / NOMINAL_TFLOPS,
                       "what": "full recompute, whole step time (all kernels) against the conv FLOPs of 4 x the n=128 step"}
            # the bandwidth kernels at the size where they are no longer launch-latency-scale (north_star: achieved HBM GB/s
            # of the snapshot and overlap-add kernels): per-kernel stamps of the same step
            order_l, acc_l = le.profile(reps=4, prewarm_s=0.3, ms_per_step=ms_l / n_l)
            kern_l, _ = kernel_table(le, order_l, acc_l, pk, (c4 or {}).get("sm_mhz") or 1700.0, sms)
            largest["bandwidth_kernels"] = {k: v for k, v in kern_l.items() if "gbs" in v}
            le.close()
            del le
        except Exception as ex:                      # e.g. a smaller box: report, do not fail the bench line
            largest = {"error": str(ex)[:300]}
        torch.cuda.empty_cache()

    # offline / non-streaming mode (D9): the same number of detector-windows per launch, but all from ONE
    # stream's archival segment (B = n windows advance the stream by B*S samples per launch)
    cs = torch.cuda.Stream()
    dtype = gw.GW_BF16 if args.dtype == "bf16" else gw.GW_FP16
    dc_params, _ = make_params(cfg)
    offline = None
    if not args.no_offline:
        B = sp.n_streams
        one = S.StreamSpec(1, sp.n_det, sp.fs, sp.window, sp.stride, sp.n_witness)
        off = gw.Offline(one, cfg.dc_layers, dc_params, B, dtype)
        seg = torch.from_numpy(synth.stream_channels(cfg.seed, one, off.samples)).cuda()
        cl = torch.empty((sp.n_det, off.samples), device="cuda")
        nz = torch.empty((sp.n_det, off.samples), device="cuda")
        with torch.cuda.stream(cs):
            for _ in range(3):
                off.run(seg, cl, nz, cs)
            o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            o0.record(cs)
            n_off = max(10, min(K, 50))
            for _ in range(n_off):
                off.run(seg, cl, nz, cs)
            o1.record(cs)
        torch.cuda.synchronize()
        off_ms = o0.elapsed_time(o1) / n_off
        offline = {"windows_per_launch": B, "samples_per_launch": off.samples, "ms_per_launch": off_ms,
                   "value": B * sp.stride / FS / (off_ms * 1e-3), "unit": UNIT,
                   "tflops_whole_launch": round(sum(a["flops"] for k, a in acc.items() if k.startswith("gemm.dc")) / (off_ms * 1e-3) / 1e12, 1),
                   "what": "gw_offline_run on a device-resident segment of one 2-detector stream; value counts the B*S new "
                           "samples a launch advances the stream by"}
        del off, seg, cl, nz

    # the snapshotter alone at the paper's highest update rates ("the bottleneck in this
    # pipeline is the streaming state update" at r = fs/3 and fs/2, i.e. strides of 3 and 2 samples; r = fs was not
    # attempted there): one stream, 44 channels, W = 32768, a ring append of `stride` samples per update
    snapshotter = None
    if not args.no_offline:
        snapshotter = {}
        for st_small in (1, 2, 3, 16):
            sps = S.StreamSpec(1, sp.n_det, sp.fs, sp.window, st_small, sp.n_witness)
            ss = gw.Stream(sps)
            new = torch.randn((1, sps.channels, st_small), device="cuda")
            n_u = 2000
            with torch.cuda.stream(cs):
                for _ in range(50):
                    ss.update(new, cs)
                s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                s0.record(cs)
                for _ in range(n_u):
                    ss.update(new, cs)
                s1.record(cs)
            torch.cuda.synchronize()
            us = 1e3 * s0.elapsed_time(s1) / n_u
            snapshotter[f"stride_{st_small}"] = {"us_per_update": round(us, 3), "updates_per_s": round(1e6 / us),
                                                 "realtime_rate_hz": FS / st_small}
            ss.close()
        snapshotter["what"] = ("gw_stream_update alone, eager launches of k_append on one stream, 2000 updates, CUDA events; "
                               "real time needs realtime_rate_hz updates per second")

    # BASELINE.json configs[2] on its own: 256 windows x 2 detectors x 4096 samples through the stateless classifier
    classifier = None
    if not args.no_offline:
        c2 = S.config_c2()
        cp2, dp2 = synth.bbh_params(c2.seed * 100 + 50, c2.bbh_convs, c2.bbh_dense)
        wins = torch.from_numpy(synth.bbh_windows(c2.seed, 256, c2.bbh_len)).cuda()
        classifier = {"windows": 256, "what": "gw_bbh_score_batch (stateless), device-resident windows, CUDA events over 50 calls; "
                                              "one_kernel = gw_options.fuse_bbh (default), three_kernels = fuse_bbh 0"}
        for name, fuse in (("one_kernel", 1), ("three_kernels", 0)):
            bb = gw.Bbh(None, c2.bbh_convs, cp2, dp2, c2.bbh_len, dtype, n_det=2, max_batch=256, opts=gw.Options(fuse_bbh=fuse))
            with torch.cuda.stream(cs):
                for _ in range(5):
                    bb.score_batch(wins, cs)
                c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                c0.record(cs)
                for _ in range(50):
                    bb.score_batch(wins, cs)
                c1.record(cs)
            torch.cuda.synchronize()
            us = 1e3 * c0.elapsed_time(c1) / 50
            classifier[name] = {"us_per_batch": round(us, 2), "windows_per_s": round(256 / (us * 1e-6)),
                                "data_seconds_per_s": round(256 * c2.bbh_len / FS / (us * 1e-6), 1)}
            bb.close()
        del wins

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        n_all = oracle.num_threads()
        times, cores = oracle_rate(cfg, args.dtype, 200, budget_s=15.0)   # a bounded sample: ~15 s of oracle time
        sec = sum(times)
        cpu = {"value": len(times) * (sp.stride / FS) / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{len(times)} consecutive updates of one 2-detector stream of the same workload ({sec:.1f} s of oracle time)",
               "note": "the fp64 direct-loop checker as it stands: a reported baseline, not a competent CPU implementation and "
                       "not a speed-up claim"}
        oracle.set_num_threads(1)
        t1, _ = oracle_rate(cfg, args.dtype, 3, budget_s=8.0)
        oracle.set_num_threads(n_all)
        cpu["single_thread"] = {"value": len(t1) * (sp.stride / FS) / sum(t1), "unit": UNIT, "cores": 1,
                                "sample": f"{len(t1)} updates ({sum(t1):.1f} s)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16" if args.dtype == "fp16" else "bf16", "data": "synthetic",
            "config": {"workload": f"C4 multi-stream ensemble (configs[4]): n={sp.n_streams} independent config-3 streams "
                                   f"per GPU, 2 detectors x 21 witnesses, W={sp.window}, S={sp.stride}, fs={FS}, "
                                   f"classifier on last {cfg.bbh_len} samples, one CUDA-graph launch per stride"
                                   + (", incremental path" if args.incremental else ", full recompute of every window"),
                       "n_streams_per_gpu": sp.n_streams, "stride": sp.stride, "window": sp.window,
                       "l2": f"inputs larger than L2: ring state {sp.n_streams * sp.channels * sp.window * 4 / 2**20:.0f} MiB "
                             "is re-read every step", "precision": f"{args.dtype} storage, fp32 accumulate"},
            "sustained": sustained, "latency": latency, "e2e": e2e, "gpu_launches": int(launches),
            "graph_nodes": graph_nodes,
            "roofline": roofline, "smem_peak_gbs": round(smem_peak_gbs, 1), "mufu": mufu, "kernels": kernels, "clocks": clocks,
            "incremental": incremental, "largest": largest, "cpu_baseline": cpu, "offline": offline, "classifier_c2": classifier, "snapshotter": snapshotter,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: n in {1, 16, 128, 512} x stride in {1/16, 1/8, 1/4 s} x {fp16, bf16}, one
    process per point (a fresh engine and allocator each time)."""
    rows = []
    for dtype in ("fp16", "bf16"):
        for n in SWEEP_STREAMS:
            for stride in SWEEP_STRIDES:
                cmd = [sys.executable, os.path.abspath(__file__), "--streams", str(n), "--stride", str(stride), "--dtype", dtype,
                       "--steps", str(args.steps), "--warmup", str(args.warmup), "--no-cpu-baseline", "--no-offline", "--no-largest",
                       "--seg-seconds", str(4 if n >= 512 else SEG_SECONDS)]
                res = subprocess.run(cmd, capture_output=True, text=True)
                line = res.stdout.strip().splitlines()[-1] if res.returncode == 0 and res.stdout.strip() else None
                if line is None:
                    log(f"sweep point n={n} S={stride} {dtype} failed:\n{res.stderr[-2000:]}")
                    continue
                with open(args.sweep, "a") as f:
                    f.write(line + "\n")
                d = json.loads(line)
                inc = d.get("incremental") or {}
                rows.append((dtype, n, stride, d["value"], d["ms_per_step"], d["latency"]["p50_ms"], d["latency"]["p99_ms"],
                             d["latency"]["realtime_budget_ms"], d["roofline"]["frac_sustained"], d["roofline"]["frac_nominal"],
                             d["e2e"]["value"], inc.get("value", float("nan")), inc.get("ms_per_step", float("nan")),
                             (inc.get("latency") or {}).get("p50_ms", float("nan")), (inc.get("latency") or {}).get("p99_ms", float("nan"))))
                log("%-5s n=%4d S=%5d  full: %9.1f data-s/s  %7.3f ms/step  p50 %7.3f  p99 %7.3f (budget %6.1f ms)  tensor %.3f of sustained %.3f of nominal  "
                    "e2e %9.1f | incremental: %9.1f data-s/s  %7.3f ms/step  p50 %7.3f  p99 %7.3f" % rows[-1])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--streams", type=int, default=128)
    ap.add_argument("--stride", type=int, default=512)
    ap.add_argument("--dtype", default="fp16", choices=["fp16", "bf16"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-pdl", action="store_true", help="disable programmatic dependent launch (A/B aid)")
    ap.add_argument("--no-snake", action="store_true", help="every layer walks its tiles forwards (A/B aid)")
    ap.add_argument("--seg-seconds", type=int, default=SEG_SECONDS, help="length of the looped input segment per stream")
    ap.add_argument("--sweep", metavar="FILE", help="run the configs[4] grid (n x stride x dtype), one bench line per "
                                                    "point appended to FILE (JSON lines); prints a table to stderr")
    ap.add_argument("--no-2sm", action="store_true", help="single-CTA kernel for the N=256 layers too (A/B aid)")
    ap.add_argument("--no-offline", action="store_true", help="skip the offline-mode measurement")
    ap.add_argument("--no-skip", action="store_true", help="issue the structurally empty MMAs too (A/B aid)")
    ap.add_argument("--incremental", action="store_true", help="time the exact incremental path as the MAIN arm (A/B aid)")
    ap.add_argument("--no-incremental", action="store_true", help="skip the incremental-path leg")
    ap.add_argument("--no-largest", action="store_true", help="skip the n=512, S=1024 point")
    ap.add_argument("--sustained-seconds", type=float, default=2.0, help="length of the back-to-back sustained leg (0: skip)")
    ap.add_argument("--timed-only", action="store_true",
                    help="only the warm-up and the timed region (for short runs under ncu); prints a reduced line")
    ap.add_argument("--reference-budget", type=float, default=150.0,
                    help="--impl reference stops after this many seconds of oracle time (a bounded sample)")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        args.warmup = min(args.warmup, 1)
        run_reference(args)
    else:
        run_native(args)


if __name__ == "__main__":
    main()
