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

    if args.no_pdl:
        gw.set_pdl(False)
    if args.no_snake:
        gw.set_snake(False)
    if args.no_skip:
        gw.set_skip_zeros(False)
    if args.no_2sm:
        gw.set_two_sm(False)
    dtype = gw.GW_BF16 if args.dtype == "bf16" else gw.GW_FP16
    cfg = S.config_c3(args.streams, args.stride, WINDOW)
    sp = cfg.stream
    n_chunks = args.seg_seconds * FS // sp.stride
    dc_params, bbh_params = make_params(cfg)
    t0 = time.time()
    chunks_h = torch.from_numpy(make_input_chunks(cfg, n_chunks)).pin_memory()
    chunks_d = chunks_h.cuda()
    log(f"[rank {rank}] inputs {tuple(chunks_h.shape)} ({chunks_h.numel() * 4 / 2**20:.0f} MiB) in {time.time() - t0:.1f}s")
    stream, dc, bbh, pipe = gw.build_ensemble(cfg, dc_params, bbh_params, dtype)
    cs = torch.cuda.Stream()
    scores = torch.zeros(sp.n_streams, device="cuda")
    final = torch.zeros((sp.n_streams, sp.n_det, sp.stride), device="cuda")
    step_no = [0]

    def step():
        pipe.step(chunks_d[step_no[0] % n_chunks], scores, final, cs)
        step_no[0] += 1

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    W_, K = max(args.warmup, 3), args.steps
    for _ in range(W_):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = gw.kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(cs)
    for _ in range(K):
        step()
    ev1.record(cs)
    barrier()
    launches = gw.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else None
    ms_total = ev0.elapsed_time(ev1)
    ms_total = shard.max_over_ranks(ms_total, device="cuda")
    ds_per_step = sp.n_streams * sp.stride / FS
    value = world * K * ds_per_step / (ms_total / 1e3)

    if args.timed_only:
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
                              "warmup": W_, "ms_per_step": ms_total / K, "gpu_launches": int(launches),
                              "note": "--timed-only run (profiling aid), not a bench line"}), flush=True)
        return

    # per-update latency: launch -> stream sync, host clock, one sample per update
    lat = []
    for _ in range(min(max(K, 50), 5000)):
        t0 = time.perf_counter()
        step()
        cs.synchronize()
        lat.append((time.perf_counter() - t0) * 1e3)
    lat.sort()
    latency = {"p50_ms": lat[len(lat) // 2], "p99_ms": lat[min(len(lat) - 1, int(len(lat) * 0.99))],
               "samples": len(lat), "per_stream_p50_ms": lat[len(lat) // 2] / sp.n_streams,
               "realtime_budget_ms": 1e3 * sp.stride / FS,
               "what": "host clock, gw_step launch -> stream synchronize, whole batch of n streams"}

    # end to end through the C ABI with HOST buffers (pinned): H2D of the new samples and D2H of the
    # scores + final cleaned samples inside the timed region, every step
    scores_h = torch.zeros(sp.n_streams).pin_memory()
    final_h = torch.zeros((sp.n_streams, sp.n_det, sp.stride)).pin_memory()
    # offline regime: gw_step_host_async, whose input copy overlaps the previous step's kernels;
    # every step's results still land in host memory inside the timed region
    for i in range(3):
        pipe.step_host_async(chunks_h[step_no[0] % n_chunks], scores_h, final_h, cs); step_no[0] += 1
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        pipe.step_host_async(chunks_h[step_no[0] % n_chunks], scores_h, final_h, cs); step_no[0] += 1
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    # online regime: gw_step_host, which returns with the results (one synchronisation per update)
    t0 = time.perf_counter()
    for _ in range(min(K, 50)):
        pipe.step_host(chunks_h[step_no[0] % n_chunks], scores_h, final_h, cs); step_no[0] += 1
    e2e_sync_ms = 1e3 * (time.perf_counter() - t0) / min(K, 50)
    e2e_s = shard.max_over_ranks(e2e_s, device="cuda")
    h2d = sp.n_streams * sp.channels * sp.stride * 4
    d2h = sp.n_streams * 4 + sp.n_streams * sp.n_det * sp.stride * 4
    e2e = {"value": world * K * ds_per_step / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * e2e_s / K,
           "ms_per_step_synchronous": e2e_sync_ms,
           "what": "gw_step_host_async: pinned host buffers, H2D of every step's samples and D2H of its scores and "
                   "final cleaned samples inside the timed region, host clock; ms_per_step_synchronous = gw_step_host "
                   "(returns with the results of each update)"}

    # per-kernel device times: eager replay of the same step with a CUDA event after every launch
    prof = {}
    n_prof = 5
    for it in range(n_prof + 1):
        rows = pipe.step_profile(chunks_d[step_no[0] % n_chunks], scores, final, cs); step_no[0] += 1
        if it == 0:
            continue
        for label, ms, fl in rows:
            a = prof.setdefault(label, [0.0, 0.0])
            a[0] += ms / n_prof
            a[1] = fl
    smem_bytes = pipe.profile_smem_bytes()
    pk = peaks()
    gemm_ms = sum(v[0] for k, v in prof.items() if k.startswith("gemm."))
    gemm_fl = sum(v[1] for k, v in prof.items() if k.startswith("gemm."))
    step_ms_eager = sum(v[0] for v in prof.values())
    achieved = gemm_fl / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get("conv_gemm_dram_bytes_per_launch")
    roofline = {"bound": "tensor", "kernel": "k_conv_gemm_umma (all conv-GEMM launches of one step)",
                "achieved": achieved, "peak": pk["tensor_tflops"], "unit": "TFLOP/s",
                "frac": achieved / pk["tensor_tflops"], "traffic": traffic, "peak_source": pk["source"],
                "flops_per_step": gemm_fl, "ms_per_step_in_kernel": gemm_ms,
                "share_of_step": gemm_ms / step_ms_eager if step_ms_eager else None,
                "timing": "CUDA events after every launch, eager replay of the same step on the launch stream"}
    kernels = {k: {"ms": round(v[0], 4), **({"tflops": round(v[1] / (v[0] * 1e-3) / 1e12, 1)} if v[1] else {})}
               for k, v in prof.items()}
    # bandwidth kernels: ALGORITHMIC bytes per step / event time
    nd, nw = sp.n_det, sp.n_witness
    hbm_bytes = {
        "append": sp.n_streams * sp.channels * sp.stride * 8,                       # read new + write ring
        "ring16_append": sp.n_streams * nd * sp.stride * (nw * 4 + 2 * 32 * 2),     # read fp32, write both mirror copies
        "snapshot_append": sp.n_streams * (sp.channels * sp.stride * 8 + nd * sp.stride * 2 * 32 * 2),  # a1 + a2 fused
        "aggregate": sp.n_streams * nd * sp.window * 20,                            # p_t, acc r/w, strain, cleaned
        "bbh_conv1": sp.n_streams * (nd * cfg.bbh_len * 4 + (cfg.bbh_len // 4) * 32 * 2),
    }
    for k, b in hbm_bytes.items():
        if k in kernels and kernels[k]["ms"] > 0:
            gbs = b / (kernels[k]["ms"] * 1e-3) / 1e9
            kernels[k].update({"gbs": round(gbs, 1), "hbm_frac": round(gbs / pk["hbm_gbs"], 3)})
    # conv GEMMs against the shared-memory operand roofline: traffic by the engine's accounting
    # (MMA operand reads + TMA fills + epilogue staging) over 128 B/clk per SM at the SM clock sampled under load
    sm_mhz = (clocks or {}).get("sm_mhz") or 1700.0
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    smem_peak_gbs = sms * 128 * sm_mhz * 1e6 / 1e9
    for k, b in smem_bytes.items():
        if k in kernels and kernels[k]["ms"] > 0:
            gbs = b / (kernels[k]["ms"] * 1e-3) / 1e9
            kernels[k].update({"smem_gbs": round(gbs, 1), "smem_frac": round(gbs / smem_peak_gbs, 3)})

    # offline / non-streaming mode (D9): the same number of detector-windows per launch, but all from ONE
    # stream's archival segment (B = n windows advance the stream by B*S samples per launch)
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
                   "tflops_whole_launch": round(sum(v[1] for k, v in prof.items() if k.startswith("gemm.dc")) / (off_ms * 1e-3) / 1e12, 1),
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

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        times, cores = oracle_rate(cfg, args.dtype, 200, budget_s=15.0)   # a bounded sample: ~15 s of oracle time
        sec = sum(times)
        cpu = {"value": len(times) * (sp.stride / FS) / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{len(times)} consecutive updates of one 2-detector stream of the same workload ({sec:.1f} s of oracle time)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W_,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16" if args.dtype == "fp16" else "bf16", "data": "synthetic",
            "config": {"workload": f"C4 multi-stream ensemble (configs[4]): n={sp.n_streams} independent config-3 streams "
                                   f"per GPU, 2 detectors x 21 witnesses, W={sp.window}, S={sp.stride}, fs={FS}, "
                                   f"classifier on last {cfg.bbh_len} samples, one CUDA-graph launch per stride",
                       "n_streams_per_gpu": sp.n_streams, "stride": sp.stride, "window": sp.window,
                       "l2": f"inputs larger than L2: ring state {sp.n_streams * sp.channels * sp.window * 4 / 2**20:.0f} MiB "
                             "is re-read every step", "precision": f"{args.dtype} storage, fp32 accumulate"},
            "latency": latency, "e2e": e2e, "gpu_launches": int(launches), "graph_nodes": pipe.graph_nodes(),
            "roofline": roofline, "smem_peak_gbs": round(smem_peak_gbs, 1), "kernels": kernels, "clocks": clocks, "cpu_baseline": cpu, "offline": offline, "snapshotter": snapshotter,
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
                       "--steps", str(args.steps), "--warmup", str(args.warmup), "--no-cpu-baseline", "--no-offline",
                       "--seg-seconds", str(4 if n >= 512 else SEG_SECONDS)]
                res = subprocess.run(cmd, capture_output=True, text=True)
                line = res.stdout.strip().splitlines()[-1] if res.returncode == 0 and res.stdout.strip() else None
                if line is None:
                    log(f"sweep point n={n} S={stride} {dtype} failed:\n{res.stderr[-2000:]}")
                    continue
                with open(args.sweep, "a") as f:
                    f.write(line + "\n")
                d = json.loads(line)
                rows.append((dtype, n, stride, d["value"], d["ms_per_step"], d["latency"]["p50_ms"], d["latency"]["p99_ms"],
                             d["latency"]["realtime_budget_ms"], d["roofline"]["frac"], d["e2e"]["value"]))
                log("%-5s n=%4d S=%5d  %9.1f data-s/s  %7.3f ms/step  p50 %7.3f  p99 %7.3f (budget %6.1f ms)  tensor %.3f  e2e %9.1f"
                    % rows[-1])


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
