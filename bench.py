#!/usr/bin/env python
"""bench.py -- decoded range-gate spectra/s of the plspec hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]
    (N > 1: python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...)

A "step" is one whole integration of the workload: plspec_accumulate over all its IPPs (sc16
conversion, decode, FFT, |X|^2, accumulation -- every row of SURVEY.md 8(a)) followed by
plspec_finalize (spectra written out once, accumulators cleared).  Default workload: cfg3 =
BASELINE.json configs[2] (N = 16384, the length the metric is quoted at).

value  : spectra/s with inputs resident in HBM, timed on the device with CUDA events,
         L2 flushed between steps, max over ranks.
e2e    : the same metric through the same C-ABI calls with HOST (pinned) buffers: the H2D copy
         of voltages + codes and the D2H copy of S are inside the timed region.
roofline: the fused kernel against the FP32 ALU roofline (5 N log2 N flops per window).
cpu_baseline: the float64 oracle on this box's host cores, on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2311_18737_b200 import synth  # noqa: E402

METRIC = "decoded range-gate spectra/s at N=16384"
UNIT = "spectra/s"
# FP32 ALU peak, derived: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz max SM clock (B200_PROFILING.md
# unit counts and clocks).  The MEASURED rate (plspec_diag_fp32_peak, run below under the
# clock sampler) is printed beside it as roofline.peak_measured.
N_SM, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
ALU_PEAK_TFLOPS = N_SM * FP32_LANES * 2 * SM_MAX_GHZ / 1e3
PAPER_BEST_SPECTRA_PER_S = 409600 / 1.488      # GTX 780 Ti, PAPER.md:139 (workload "paper" only)


def metric_name(w):
    return METRIC if w.N == 16384 else f"decoded range-gate spectra/s at N={w.N}"


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region: NVML polled from a thread
    (about 1 ms per sample, so even the 5 ms cfg-2 region is covered); nvidia-smi -lms as a fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None
        self.nvml, self.handle, self.samples, self.run, self.source = None, None, [], False, None

    def _nvml_open(self):
        import pynvml
        import torch
        pynvml.nvmlInit()
        uuid = str(torch.cuda.get_device_properties(self.index).uuid)
        if not uuid.startswith("GPU-"):
            uuid = "GPU-" + uuid
        self.handle = pynvml.nvmlDeviceGetHandleByUUID(uuid)
        self.nvml = pynvml
        self.mx = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        self.masks = [(n, getattr(pynvml, a)) for n, a in zip(self.NAMES, (
            "nvmlClocksThrottleReasonHwSlowdown", "nvmlClocksThrottleReasonHwThermalSlowdown",
            "nvmlClocksThrottleReasonSwThermalSlowdown", "nvmlClocksThrottleReasonSwPowerCap"))]

    def _poll(self):
        nv, h = self.nvml, self.handle
        while self.run:
            try:
                self.samples.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                     nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                                     int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))))
            except Exception:
                pass
            time.sleep(0.0005)

    def start(self):
        try:
            self._nvml_open()
            self.run, self.source = True, "nvml"
            self.t = threading.Thread(target=self._poll, daemon=True)
            self.t.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi"
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        sm, mx, pw, reasons = [], [], [], set()
        if self.nvml:
            self.run = False
            self.t.join(timeout=2)
            for c, p, r in self.samples:
                sm.append(c); mx.append(self.mx); pw.append(p)
                reasons.update(n for n, m in self.masks if r & m)
        elif self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
            for ln in self.lines:
                f = [x.strip() for x in ln.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
                except ValueError:
                    continue
                for n, v in zip(self.NAMES, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        else:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml and nvidia-smi unavailable"]}
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_min_mhz": float(min(sm)), "sm_max_mhz": float(max(mx)),
                "power_w_max": float(max(pw)), "samples": len(sm), "source": self.source, "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def cpu_oracle_sample(w, V, C, target_s=12.0, steps=1):
    """Time the oracle as it stands on a bounded sample: a subset of gates over ALL IPPs
    (gates are independent and cost the same, so the rate extrapolates exactly)."""
    import oracle
    cores = oracle.max_threads()
    # calibrate with all threads busy: `cores` gates x a few IPPs
    pc = min(4, w.n_ipp)
    for _ in range(2):                                           # the first call also starts the OpenMP team
        t0 = time.perf_counter()
        oracle.spectra(V[:pc], C[:pc], N=w.N, n_ranges=min(cores, w.n_ranges), r0=w.r0, stride=w.stride)
        per_round = (time.perf_counter() - t0) / pc * w.n_ipp    # seconds for `cores` gates x all IPPs
    rounds = int(max(1, target_s / max(per_round, 1e-9)))
    gates = min(w.n_ranges, rounds * cores)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        oracle.spectra(V, C, N=w.N, n_ranges=gates, r0=w.r0, stride=w.stride)
        times.append(time.perf_counter() - t0)
    dt = float(np.mean(times))
    return {"value": gates * w.n_ipp / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{gates} of {w.n_ranges} gates x all {w.n_ipp} IPPs of {w.name} "
                      f"({gates * w.n_ipp} windows, {dt:.1f} s per step, float64 radix-2, OpenMP over gates)"}, dt


def cufft_pipeline(w, V_dev, C_dev, steps, flush):
    """Comparison point, not the product (north_star): the unfused structure the paper describes
    as written -- per pulse a "complex multiplication" kernel that writes `batch[R][N]` to device memory, one
    in-place batched cufftExecC2C over its rows (cufftPlanMany), and a "spectrum accumulation" kernel -- built
    from csrc/cufft_pipeline.cu into libplspec_cufft.so, on the same device-resident inputs and timed with CUDA
    events like `value` (spectrum zeroed inside the timed region, as finalize does for ours)."""
    import ctypes
    import torch
    from paper_2311_18737_b200 import build as plbuild
    L = ctypes.CDLL(plbuild.build_cufft_pipeline())
    vp, ci = ctypes.c_void_p, ctypes.c_int
    L.plspec_cufft_create.argtypes = [ci, ci, ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
    L.plspec_cufft_accumulate.argtypes = [vp, vp, vp, ci, vp, vp]
    L.plspec_cufft_launches.argtypes = [vp]
    L.plspec_cufft_launches.restype = ctypes.c_longlong
    L.plspec_cufft_destroy.argtypes = [vp]
    h = vp()
    rc = L.plspec_cufft_create(w.N, w.code_len, w.n_ranges, w.r0, w.stride, w.ipp_len, w.dtype, ctypes.byref(h))
    if rc != 0:
        raise RuntimeError(f"plspec_cufft_create failed ({rc})")
    S = torch.zeros((w.n_ranges, w.N), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream

    def step():
        S.zero_()
        rc = L.plspec_cufft_accumulate(h, V_dev.data_ptr(), C_dev.data_ptr(), w.n_ipp, S.data_ptr(), stream)
        if rc != 0:
            raise RuntimeError(f"plspec_cufft_accumulate failed ({rc})")

    try:
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        ms = []
        for _ in range(steps):
            flush.fill_(4)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            step()
            e1.record()
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
    finally:
        L.plspec_cufft_destroy(h)
    return float(np.mean(ms)), S


def ncu_traffic(name):
    """DRAM bytes per fused-kernel launch from the committed `ncu --set full` capture of this workload
    (dram__bytes_read.sum + dram__bytes_write.sum), with the capture it came from; (None, why) if there is none.
    The table sits beside the binding (paper_2311_18737_b200/ncu_traffic.json) and is refreshed by hand from
    profiles/ whenever the kernels change: a number from a profiler run is evidence, never a bench value."""
    try:
        t = json.load(open(os.path.join(ROOT, "paper_2311_18737_b200", "ncu_traffic.json")))
        e = t["workloads"].get(name)
        if e:
            return int(e["dram_bytes_per_launch"]), e["source"]
        return None, "no ncu capture of this workload committed"
    except Exception as e:
        return None, f"ncu_traffic.json unreadable: {type(e).__name__}"


def products_timing(w, S_dev, flush, reps=7, it=None, accumulate=None):
    """plspec_mean_spectrum (centred) and plspec_profile on the finished S: median of `reps` launches, L2 flushed
    before each, CUDA events on the current stream.  Both are one pass over S: algorithmic bytes 8 and 4 per bin,
    against the measured HBM copy peak (MEASURED_PEAKS.json, else the profiling guide's 6 550 GB/s fallback)."""
    import torch
    from paper_2311_18737_b200 import binding as pl
    R, N = w.n_ranges, w.N
    try:
        peak, src = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json"
    except Exception:
        peak, src = 6550.0, "fallback (B200_PROFILING.md)"
    P = torch.empty_like(S_dev)
    ki = torch.empty((2, R), dtype=torch.int32, device="cuda"); pf = torch.empty((3, R), dtype=torch.float32, device="cuda")
    # These kernels are HBM-bound and last tens of microseconds.  After the write flush L2 is full of DIRTY lines whose
    # write-back would be charged to the kernel that evicts them, so the write flush is followed by a read of a second
    # buffer larger than L2: the kernel then starts from a cache of clean lines that hold none of its data.
    clean = torch.zeros(flush.numel() // 4, dtype=torch.int32, device="cuda")

    def flush_l2():
        flush.fill_(3)
        clean.sum()

    calls = {"mean_spectrum_centred": (8, lambda: pl.plspec_mean_spectrum(S_dev, P, R, N, w.n_ipp, True)),
             "profile": (4, lambda: pl.plspec_profile(S_dev, R, N, w.n_ipp, max(1, N // 256), 2, ki[0], pf[0], ki[1],
                                                      pf[1], pf[2]))}
    out = {"hbm_peak_gbs": peak, "peak_source": src}
    # two yardsticks under the very same timing: the smallest launch this library has (plspec_profile of one 16-bin
    # gate: what the two events see of a launch that moves nothing) and a plain library pass over S (torch.sum: 4 B per
    # bin, no search): context for what a one-pass product of this size can reach between two events
    S1 = torch.ones((1, 16), dtype=torch.float32, device="cuda")
    calls["empty_launch"] = (0, lambda: pl.plspec_profile(S1, 1, 16, 1, 1, 0, ki[0], pf[0], ki[1], pf[1], pf[2]))
    calls["read_pass_torch_sum"] = (4, lambda: S_dev.sum())
    for name, (bpb, call) in calls.items():
        ts = []
        for _ in range(reps + 2):
            flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); call(); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms = float(np.median(ts[2:]))
        gbs = bpb * R * N / ms / 1e6
        out[name] = {"ms": ms, "bytes_per_bin": bpb, "GB/s": gbs, "frac": gbs / peak}
    if it is not None:
        # the write-out alone (plspec_finalize to device memory: 12 B per bin -- accumulators read and zeroed, S_out
        # written) against the write-out with both products folded in (plspec_finalize_products: 16 B per bin, P_out
        # besides; the stand-alone sequence finalize + mean + profile moves 24 B per bin); each after a fresh
        # integration, L2 flushed, the blocking call between two events
        k_min = max(1, N // 256)
        fin = {"finalize": (12, lambda: it.finalize(S_dev)),
               "finalize_products": (16, lambda: it.finalize_products(S_dev, w.n_ipp, P_out=P, centred=True, k_min=k_min, guard=2,
                                                                      k_up=ki[0], p_up=pf[0], k_dn=ki[1], p_dn=pf[1],
                                                                      noise=pf[2]))}
        for name, (bpb, call) in fin.items():
            ts = []
            for _ in range(5):
                accumulate()
                torch.cuda.synchronize()
                flush_l2()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); call(); e1.record()
                torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            ms = float(np.median(ts[1:]))
            gbs = bpb * R * N / ms / 1e6
            out[name] = {"ms": ms, "bytes_per_bin": bpb, "GB/s": gbs, "frac": gbs / peak}
    return out


def workload_config(w, l2, parallelism):
    """The `config` object of the JSON line: what defines the workload, the same keys for both arms."""
    return {"workload": w.name, "N": w.N, "code_len": w.code_len, "n_ranges": w.n_ranges, "stride": w.stride,
            "n_ipp": w.n_ipp, "ipp_len": w.ipp_len, "input": "sc16" if w.dtype == synth.SC16 else "complex64",
            "windows_per_step": w.windows, "l2": l2, "parallelism": parallelism}


def run_reference(args, w):
    """--impl reference: the oracle (the only 'reference implementation' this tier has), as it stands, on the
    host cores.  Every one of the `warmup` + `steps` steps is run; each is a bounded sample of the workload (a
    subset of gates over all IPPs) sized so that the whole run ends within about two minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    V, C = synth.make_inputs(w)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    per_step_s = min(10.0, 110.0 / (steps + warmup))
    if warmup:
        cpu_oracle_sample(w, V, C, target_s=per_step_s, steps=warmup)
    cb, dt = cpu_oracle_sample(w, V, C, target_s=per_step_s, steps=steps)
    line = {
        "impl": "reference", "metric": metric_name(w), "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, "n/a (float64 oracle on the host cores)",
                                  "oracle on rank 0's host cores (OpenMP over range gates)"),
        "sample_note": "each step is a bounded sample of the workload (subset of gates, all IPPs); value = windows "
                       "of the sample / its time",
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def probe_mem():
    """what an SM and the chip can move to and from L2 / DRAM (GB/s, 128-bit accesses)."""
    import torch
    from paper_2311_18737_b200 import binding as pl
    torch.cuda.set_device(0)
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    kinds = {"read": 0, "write": 1, "copy": 2, "tma_store": 3}
    out = {"probe": "plspec_diag_mem_bandwidth", "unit": "GB/s", "n_sm": n_sm, "rows": []}
    for mb, passes in ((32, 64), (64, 32), (2048, 2)):
        for ctas in (1, 8, n_sm, 2 * n_sm, 4 * n_sm):
            if mb == 2048 and ctas < n_sm:
                continue
            row = {"buffer_MiB": mb, "ctas": ctas}
            for name, kind in kinds.items():
                p = max(1, passes // 16) if ctas < n_sm else passes
                row[name] = round(pl.plspec_diag_mem_bandwidth(kind, mb << 20, ctas, p), 1)
            out["rows"].append(row)
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT comparison pipeline")
    ap.add_argument("--no-peak", action="store_true", help="skip the FP32 peak micro-benchmark")
    ap.add_argument("--probe-mem", action="store_true",
                    help="print the device's streaming bandwidths (plspec_diag_mem_bandwidth: L2-resident and DRAM-sized "
                         "buffers, reads / writes / copy / TMA stores, 1 ... 4 CTAs per SM) as one JSON line and exit")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 generic, 2 fused")
    ap.add_argument("--chunks", type=int, default=0)
    ap.add_argument("--shard", default="replicas", choices=["replicas", "ipp", "gates"],
                    help="N > 1: independent integrations (weak scaling, no collective; default), or ONE "
                         "integration sharded by IPP (sum all-reduce of S) / by range gate (all-gather)")
    ap.add_argument("--split", type=int, default=1, help="N > 16384: 1 decode pre-pass + device scratch (default), 2 ring "
                    "through L2 (one cooperative launch), 0 fully fused")
    ap.add_argument("--ring-depth", type=int, default=0, help="N > 16384, ring: steps the ring holds (0 = library default)")
    ap.add_argument("--ring-ahead", type=int, default=0, help="N > 16384, ring: steps decoded ahead (0 = library default)")
    ap.add_argument("--stage", type=int, default=1, help="1 shared-memory voltage stage where gates share samples, 2 wherever it fits, 0 direct loads")
    ap.add_argument("--shared-code", action="store_true",
                    help="workloads whose code repeats every IPP (cfg4's chirp): pass the one code (PLSPEC_OPT_SHARED_CODE)")
    ap.add_argument("--n-ipp", type=int, default=0, help="experiments: override the workload's IPP count")
    ap.add_argument("--n-ranges", type=int, default=0, help="experiments: override the workload's gate count")
    ap.add_argument("--input", default="", choices=["", "sc16", "complex64"],
                    help="experiments: override the workload's voltage dtype")
    args = ap.parse_args()
    w = synth.CONFIGS[args.workload]
    if args.n_ipp or args.n_ranges:
        w = synth.scaled(w, n_ranges=args.n_ranges or None, n_ipp=args.n_ipp or None, ipp_len=w.ipp_len)
    if args.input:
        from dataclasses import replace
        w = replace(w, dtype=synth.SC16 if args.input == "sc16" else synth.CF32,
                    sigma=1000.0 if args.input == "sc16" and w.dtype != synth.SC16 else w.sigma)
    if args.impl == "reference":
        return run_reference(args, w)
    if args.probe_mem:
        return probe_mem()
    args.warmup = max(args.warmup, 3)

    import torch
    from paper_2311_18737_b200 import binding as pl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the plspec path has no CPU fallback")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: every rank integrates its own batch of the same shape (weak scaling, no
    # data-path collective: integrations are independent problems).
    from paper_2311_18737_b200 import shard
    mode = args.shard if world > 1 else "replicas"
    wr = synth.Workload(**{**w.__dict__, "seed": w.seed + (17 * rank if mode == "replicas" else 0)})
    V_np, C_np = synth.make_inputs(wr, full_ranges=w.n_ranges)
    n_ipp_local, rows_local, r0_local = w.n_ipp, w.n_ranges, w.r0
    if mode == "ipp":                                   # this rank's IPPs of the one integration
        a, b = shard.split(w.n_ipp, rank, world)
        V_np, C_np, n_ipp_local = V_np[a:b], C_np[a:b], b - a
    elif mode == "gates":                               # this rank's gates; inputs replicated
        gs = shard.gate_shard(w.n_ranges, w.r0, w.stride, w.code_len, rank, world)
        rows_local, r0_local = gs.n_ranges, gs.r0
    V_pin = torch.from_numpy(np.ascontiguousarray(V_np)).pin_memory()
    shared_code = bool(args.shared_code)
    if shared_code and not (C_np == C_np[:1]).all():
        raise SystemExit(f"--shared-code: the codes of {w.name} differ from IPP to IPP")
    C_pin = torch.from_numpy(np.ascontiguousarray(C_np[0] if shared_code else C_np)).pin_memory()
    V_dev, C_dev = V_pin.cuda(), C_pin.cuda()
    S_dev = torch.empty((rows_local, w.N), dtype=torch.float32, device="cuda")
    S_pin = torch.empty((rows_local, w.N), dtype=torch.float32).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    it = pl.Integrator(w.N, w.code_len, rows_local, r0_local, w.stride, w.ipp_len, w.dtype, kernel=args.kernel,
                       ipp_chunks=args.chunks, stage=args.stage, split=args.split, shared_code=int(shared_code),
                       ring_depth=args.ring_depth, ring_ahead=args.ring_ahead)

    def exchange(S):
        if mode == "ipp":
            return shard.sum_spectra(S)                 # the path's one exchange step (NCCL all-reduce)
        if mode == "gates":
            return shard.gather_gates(S, w.n_ranges)
        return S

    def step_device(ev=None):
        if ev:
            ev[0].record()
        it.accumulate(V_dev, C_dev, n_ipp_local)
        if ev:
            ev[1].record()
        it.finalize(S_dev)
        exchange(S_dev)

    def step_host():
        it.accumulate(V_pin, C_pin, n_ipp_local)
        it.finalize(S_pin)
        if mode != "replicas":
            exchange(S_pin.cuda())

    # ---- measured FP32 multiply-add peak (the roofline's measured denominator), clocks sampled meanwhile
    peak_meas = None
    if rank == 0 and not args.no_peak:
        ps = ClockSampler(local)
        ps.start()
        pk2 = pl.plspec_diag_fp32_peak(packed=True, iters=1 << 16, reps=40)     # FFMA2: what the fused kernel issues
        pk1 = pl.plspec_diag_fp32_peak(packed=False, iters=1 << 16, reps=40)    # scalar FFMA
        pc = ps.stop()
        peak_meas = {"ffma2_tflops_best": pk2["tflops_best"], "ffma2_tflops_mean": pk2["tflops_mean"],
                     "ffma_tflops_best": pk1["tflops_best"], "ffma_tflops_mean": pk1["tflops_mean"], "clocks": pc,
                     "how": "plspec_diag_fp32_peak: 4 x 512 threads per SM, 32 independent multiply-add chains per "
                            "thread, 40 launches of 65536 iterations each, CUDA events"}

    # ---- device-resident timing
    for _ in range(args.warmup):
        flush.fill_(1)
        step_device()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = it.stats()["kernel_launches"]
    step_ms, kern_ms = [], []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.fill_(2)                                              # L2 flush, outside the event pair
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step_device((k0, k1))
        e1.record()
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        kern_ms.append(k0.elapsed_time(k1))
    barrier()
    wall_s = time.perf_counter() - t_wall0
    launches = it.stats()["kernel_launches"] - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = float(np.sum(step_ms))
    stats = it.stats()

    # ---- end to end: host pinned inputs -> S on the host
    e2e_ms = None
    if not args.no_e2e:
        for _ in range(2):
            step_host()
        barrier()
        ts = []
        for _ in range(args.steps):
            flush.fill_(3)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            step_host()                                             # finalize blocks until S_pin is complete
            ts.append((time.perf_counter() - t0) * 1e3)
        e2e_ms = float(np.sum(ts))
        barrier()

    # ---- comparison point: unfused cuFFT pipeline (rank 0, N = 1 only)
    cufft = None
    if world == 1 and not args.no_cufft:
        try:
            cms, S_cu = cufft_pipeline(w, V_dev, C_dev.expand(w.n_ipp, -1).contiguous() if shared_code else C_dev,
                                       max(1, min(args.steps, 3)), flush)
            step_device()
            ref = S_cu.mean(dim=1, keepdim=True)
            dev = float(((S_dev - S_cu).abs() / ref).max())
            decoded = w.windows * w.N
            cufft = {"ms_per_step": cms, "value": w.windows / (cms * 1e-3), "unit": UNIT,
                     "max_rel_dev_vs_fused": dev,
                     "model_dram_bytes_per_decoded_sample": 40, "model_ms_at_hbm_peak": decoded * 40 / 6.55e12 * 1e3,
                     "kind": "csrc/cufft_pipeline.cu: complex_multiplication_kernel -> cufftPlanMany/cufftExecC2C "
                             "in place over batch[R][N] -> spectrum_accumulation_kernel, looped per pulse "
                             "(PAPER.md:105-121); device-resident inputs"}
            del S_cu
        except Exception as e:                                      # comparison only: never fails the bench
            cufft = {"error": f"{type(e).__name__}: {e}"[:200]}

    # ---- post-integration products on the finished spectrum (outside the timed region)
    products = None
    if world == 1:
        try:
            products = products_timing(w, S_dev, flush, it=it if mode == "replicas" else None,
                                       accumulate=lambda: it.accumulate(V_dev, C_dev, n_ipp_local))
        except Exception as e:                                      # reported beside the metric: never fails the bench
            products = {"error": f"{type(e).__name__}: {e}"[:200]}

    # ---- max over ranks
    total_ms, e2e_max, kern_mean = shard.max_over_ranks([total_ms, e2e_ms or 0.0, float(np.mean(kern_ms))],
                                                        device="cuda")
    e2e_ms = e2e_max if e2e_ms is not None else None

    if rank == 0:
        windows_per_step = w.windows * (world if mode == "replicas" else 1)
        value = windows_per_step * args.steps / (total_ms * 1e-3)
        esz = 4 if w.dtype == synth.SC16 else 8
        h2d = w.n_ipp * w.span * esz + (1 if shared_code else w.n_ipp) * w.code_len * 8
        # one launch of a sharded integration transforms this rank's share of the windows (kern_mean is the
        # max over ranks of one rank's time); replicas each transform the whole workload
        share = (n_ipp_local / w.n_ipp) * (rows_local / w.n_ranges)
        flops_per_launch = w.fft_flops * share                      # 5 N log2 N x windows of one launch
        achieved = flops_per_launch / (kern_mean * 1e-3) / 1e12
        traffic, traffic_source = ncu_traffic(w.name) if share == 1.0 else (None, "sharded launch: not captured")
        line = {
            "metric": metric_name(w), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak" if mode == "replicas" else "strong",
            "vs_baseline": (value / PAPER_BEST_SPECTRA_PER_S) if w.name == "paper" else None,
            "dtype": "f32", "data": "synthetic",
            "config": workload_config(w, "flushed between steps (256 MB write)",
                                      (f"{world} independent integrations (one per GPU)" if mode == "replicas" else
                                       f"one integration sharded by {mode} over {world} GPUs")),
            "impl_detail": {"kernel": {1: "generic", 2: "fused"}[stats["kernel_kind"]],
                            "ipp_chunks": stats["ipp_chunks_last"], "shared_code": shared_code},
            "realtime_factor": w.data_seconds * (world if mode == "replicas" else 1) * args.steps / (total_ms * 1e-3),
            "wall_s_timed_region": wall_s,
            "clocks": clocks,
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / ALU_PEAK_TFLOPS, "traffic": traffic, "traffic_source": traffic_source,
                         "kernel": "fused_kernel" if stats["kernel_kind"] == 2 else "generic_kernel",
                         "kernel_ms": kern_mean, "flops_per_launch": flops_per_launch,
                         "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md); "
                                        "MEASURED_PEAKS.json holds no FP32 ALU figure",
                         "hbm_bytes_algorithmic": int((n_ipp_local * (w.ipp_len * esz + w.code_len * 8)
                                                       + rows_local * w.N * 4))},
        }
        if peak_meas is not None:
            pm = peak_meas["ffma2_tflops_mean"]
            line["roofline"].update({
                "peak_measured": pm, "frac_of_measured": achieved / pm,
                "peak_clock_mhz": peak_meas["clocks"].get("sm_mhz"), "peak_measurement": peak_meas})
        if e2e_ms is not None:
            line["e2e"] = {"value": windows_per_step * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                           "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(w.n_ranges * w.N * 4),
                           "ms_per_step": e2e_ms / args.steps,
                           "realtime_factor": w.data_seconds * (world if mode == "replicas" else 1) * args.steps
                                              / (e2e_ms * 1e-3)}
        if cufft is not None:
            line["cufft_pipeline"] = cufft
        if products is not None:
            line["products"] = products
        if world == 1 and not args.no_cpu_baseline:
            cb, _ = cpu_oracle_sample(w, V_np, C_np)
            line["cpu_baseline"] = cb
        print(json.dumps(line), flush=True)
    it.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
