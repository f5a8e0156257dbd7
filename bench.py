#!/usr/bin/env python
"""bench.py -- throughput of the FP8 attention forward hot path on B200 (contract: task prompt).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg4-fp8|cfg4-bf16|cfg5]
                    [--impl ours|reference] [--no-extra]

A step is one fp8attn_fwd call (the whole hot path: staging, QK^T, online softmax, P-cast,
P.V, epilogue; plus the combine kernel for split-KV decode) over one synthetic batch of the
named BASELINE.json config.  Default workload: cfg3 (configs[2]), the configuration the
"FP8 attn fwd TFLOPS" metric is quoted on; cfg4 in FP8 mode, cfg4 in BF16 isolation mode and cfg5
(decode, GB/s) are measured beside it and reported under "extra" unless --no-extra.

`value` is device-timed with inputs resident in HBM; `e2e` goes through fp8attn_fwd_host with
pinned host buffers (H2D of q,k,v and D2H of o inside the timed region).  `--impl reference`
times the CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
Inputs (403 MB of E4M3 q,k,v + 537 MB of o at cfg3; 4.3 GB of KV cache at cfg5) are larger
than the 126 MB L2, so no L2 flush is needed between timed iterations.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_06521_b200 import workloads as W   # noqa: E402  (no CUDA, no arithmetic)

WORKLOADS = {
    # name: (config, input kind, P mode, S, kv_order)
    "cfg3": ("cfg3", "e4m3", 2, 256.0, 1),
    "cfg4-fp8": ("cfg4", "e4m3", 2, 256.0, 1),
    "cfg4-bf16": ("cfg4", "bf16", 1, 256.0, 1),
    "cfg5": ("cfg5", "decode", 2, 256.0, 1),
}


# tiling the library uses for each workload (block_m, block_n, num_splits); the reference arm mirrors it so that both
# arms describe the same configuration (the oracle takes block_n and the split bounds from here)
TILING = {"cfg3": (256, 128, 1), "cfg4-fp8": (256, 128, 1), "cfg4-bf16": (256, 128, 1), "cfg5": (128, 128, 4)}


def config_of(workload, block_m, block_n, num_splits):
    cfg_name, kind, mode, S, order = WORKLOADS[workload]
    cfg = W.CONFIGS[cfg_name]
    return {"workload": f"{workload}: B={cfg.B} Hq={cfg.Hq} Hkv={cfg.Hkv} Lq={cfg.Lq} Lk={cfg.Lk} d={cfg.d} "
                        f"causal={cfg.causal} Delta={cfg.delta} S={S} order={'reverse' if order else 'forward'} "
                        f"mode={mode} inputs={kind}",
            "block_m": block_m, "block_n": block_n, "num_splits": num_splits,
            "l2": "inputs larger than L2 (no flush)", "sharding": "one replica of the workload per GPU"}


def load_peaks():
    """Measured peaks (driver-written MEASURED_PEAKS.json) or the profiling guide's fallback, plus the dense FP8
    GEMM peak measured on this pool in round 2 (profiles/fp8_peak.json; SURVEY.md 8(d) "FP8 peak -- measure")."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        m = json.load(open(p))
        out = {"hbm_gbs": m["hbm_gbs"], "bf16_tflops": m["bf16_tflops"],
               "bf16_tflops_sustained": m.get("bf16_tflops_sustained", m["bf16_tflops"]), "source": "measured"}
    else:
        out = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}
    try:
        out["fp8"] = json.load(open(os.path.join(ROOT, "profiles", "fp8_peak.json")))
    except (OSError, ValueError):
        out["fp8"] = None
    return out


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the committed
    `ncu --set full` capture of this workload (profiles/traffic.json; null if none was taken)."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        e = t.get(workload, {})
        return e.get("dram_bytes_per_launch") if e.get("kernel") == kernel else None
    except (OSError, ValueError):
        return None


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """SM clock / throttle-reason samples while the GPU is under load: NVML every 5 ms from a thread (falls back to
    an `nvidia-smi -lms 20` child process).  mark_start / mark_end bracket the timed region; the summary covers the
    samples taken between them (`samples`) and says how many of those fell inside the CUDA-event-timed steps."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.samples = index, None, []     # (t, sm_mhz, max_mhz, reasons)
        self.t_lo = self.t_hi = None
        self.stop = False
        self.nvml = None

    def _nvml_loop(self):
        n = self.nvml
        h = n.nvmlDeviceGetHandleByIndex(self.index)
        mx = float(n.nvmlDeviceGetMaxClockInfo(h, n.NVML_CLOCK_SM))
        bits = {"hw_slowdown": n.nvmlClocksEventReasonHwSlowdown, "hw_thermal_slowdown": n.nvmlClocksEventReasonHwThermalSlowdown,
                "sw_thermal_slowdown": n.nvmlClocksEventReasonSwThermalSlowdown, "sw_power_cap": n.nvmlClocksEventReasonSwPowerCap}
        while not self.stop:
            try:
                sm = float(n.nvmlDeviceGetClockInfo(h, n.NVML_CLOCK_SM))
                r = n.nvmlDeviceGetCurrentClocksEventReasons(h)
                self.samples.append((time.time(), sm, mx, tuple(k for k, b in bits.items() if r & b)))
            except Exception:
                pass
            time.sleep(0.005)

    def _smi_loop(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.proc.stdout:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                self.samples.append((time.time(), float(f[0]), float(f[1]),
                                     tuple(n for n, val in zip(names, f[3:7]) if val.lower().startswith("active"))))
            except ValueError:
                continue

    def __enter__(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.t = threading.Thread(target=self._nvml_loop, daemon=True)
            self.t.start()
        except Exception:
            self.nvml = None
            try:
                self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                              "--format=csv,noheader,nounits", "-lms", "20"],
                                             stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
                self.t = threading.Thread(target=self._smi_loop, daemon=True)
                self.t.start()
            except OSError:
                self.proc = None
        return self

    def mark_start(self):
        """Load starts: wait for the sampler's first sample (nvidia-smi takes a moment to come up)."""
        t0 = time.time()
        while (self.nvml or self.proc) and not self.samples and time.time() - t0 < 3.0:
            time.sleep(0.005)
        self.t_lo = time.time()

    def mark_end(self):
        self.t_hi = time.time()

    def __exit__(self, *a):
        self.stop = True
        if self.proc:
            time.sleep(0.05)
            self.proc.terminate()
        if self.nvml or self.proc:
            self.t.join(timeout=2)

    def summary(self, timed=None):
        """timed = (t0, t1): wall-clock window of the CUDA-event-timed steps, counted separately."""
        sel = [x for x in self.samples if self.t_lo is None or (self.t_lo <= x[0] <= (self.t_hi or x[0]))]
        if not sel:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        reasons = sorted({r for x in sel for r in x[3]})
        out = {"sm_mhz": float(np.median([x[1] for x in sel])), "sm_max_mhz": float(max(x[2] for x in sel)),
               "reasons": reasons, "samples": len(sel), "source": "nvml 5 ms" if self.nvml else "nvidia-smi -lms 20"}
        if timed is not None:
            out["samples_in_timed_steps"] = sum(1 for x in sel if timed[0] <= x[0] <= timed[1])
        return out


# --------------------------------------------------------------------------- workload
def units(cfg, kind):
    """(amount of the metric's unit one step processes, unit name, algorithmic figure for the roofline)."""
    if cfg.name == "cfg5":
        kv = 2.0 * cfg.B * cfg.Hkv * cfg.Lk * cfg.d            # E4M3 K and V, every byte once
        io = cfg.B * cfg.Hq * cfg.Lq * cfg.d * (2 + 4)          # BF16 q in, FP32 o out
        return (kv + io) / 1e9, "GB/s", "hbm"
    return cfg.flops / 1e12, "TFLOP/s", "tensor"


def build_device_workload(cfg, kind, seed, dev):
    """Seeded synthetic inputs (workloads.batch_qkv), one batch element at a time: generate on the
    host, upload, convert to the input dtype on the device (E4M3: fp8attn_quantize_e4m3)."""
    import torch
    from paper_2606_06521_b200 import fp8attn as fa
    e4_q = kind == "e4m3"
    e4_kv = kind in ("e4m3", "decode")
    qd = torch.uint8 if e4_q else torch.bfloat16
    kvd = torch.uint8 if e4_kv else torch.bfloat16
    q = torch.empty((cfg.B, cfg.Hq, cfg.Lq, cfg.d), dtype=qd, device=dev)
    k = torch.empty((cfg.B, cfg.Hkv, cfg.Lk, cfg.d), dtype=kvd, device=dev)
    v = torch.empty_like(k)
    sc = {}
    if e4_q:
        sc["q_scale"] = torch.empty((cfg.B, cfg.Hq), dtype=torch.float32, device=dev)
    if e4_kv:
        sc["k_scale"] = torch.empty((cfg.B, cfg.Hkv), dtype=torch.float32, device=dev)
        sc["v_scale"] = torch.empty((cfg.B, cfg.Hkv), dtype=torch.float32, device=dev)
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        futs = [ex.submit(W.batch_qkv, cfg, b, seed) for b in range(cfg.B)]
        for b, f in enumerate(futs):
            qb, kb, vb = (torch.from_numpy(a).to(dev) for a in f.result())
            futs[b] = None
            for name, src, dst, e4 in (("q", qb, q, e4_q), ("k", kb, k, e4_kv), ("v", vb, v, e4_kv)):
                if e4:
                    codes, s = fa.quantize_e4m3(src.unsqueeze(0))
                    dst[b].copy_(codes[0])
                    sc[name + "_scale"][b].copy_(s[0])
                else:
                    dst[b].copy_(src)          # FP32 -> BF16, round to nearest even
            del qb, kb, vb
    torch.cuda.synchronize()
    return q, k, v, sc


def timed_steps(step, steps, warmup, dev, world=1, min_load_s=0.5):
    """`warmup` untimed steps, then exactly `steps` steps timed with CUDA events on the current stream between
    synchronisations (a barrier before, for N > 1).  The clock sampler runs from the first timed step on; if the
    timed region is shorter than `min_load_s`, the same step keeps running (untimed) until then, so that the clock
    record holds enough samples under the same load.  Returns (per-step ms, total ms, clocks, last result)."""
    import torch
    import torch.distributed as dist
    with ClockSampler(dev.index or 0) as clk:
        for _ in range(max(warmup, 3)):
            r = step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        torch.cuda.synchronize()
        clk.mark_start()
        t0 = time.time()
        ev[0].record()
        for i in range(steps):
            r = step()
            ev[i + 1].record()
        torch.cuda.synchronize()
        t1 = time.time()
        while time.time() - t0 < min_load_s:
            for _ in range(8):
                step()
            torch.cuda.synchronize()
        clk.mark_end()
    per_step = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]
    return per_step, ev[0].elapsed_time(ev[steps]), clk.summary(timed=(t0, t1)), r


def roofline_of(workload, cfg, mode, bound, amount, kern_ms, kernel_id, peaks):
    """The roofline object of one workload: achieved = algorithmic FLOP (or bytes) per launch / measured launch time;
    peak = the measured number for a kernel timed on its own (burst), the sustained one and my own FP8 GEMM
    measurement beside it."""
    if bound == "tensor":
        is_fp8 = mode == 2
        mult = 2.0 if is_fp8 else 1.0
        roof = {"bound": "tensor", "achieved": amount / (kern_ms * 1e-3), "peak": peaks["bf16_tflops"] * mult, "unit": "TFLOP/s",
                "peak_source": f"{peaks['source']} cuBLAS bf16 burst {peaks['bf16_tflops']} TFLOP/s"
                               + (" x2 (guide's nominal fp8:bf16 ratio)" if is_fp8 else "")
                               + "; burst, not sustained: the kernel is timed on its own at full clocks",
                "peak_sustained": peaks["bf16_tflops_sustained"] * mult}
        roof["frac_vs_sustained"] = roof["achieved"] / roof["peak_sustained"]
        fp8 = peaks.get("fp8")
        if is_fp8 and fp8:
            roof["peak_measured_fp8"] = fp8["fp8_burst_tflops"]
            roof["frac_vs_measured_fp8"] = roof["achieved"] / fp8["fp8_burst_tflops"]
            roof["frac_vs_measured_fp8_sustained"] = roof["achieved"] / fp8["fp8_sustained_tflops"]
            roof["peak_measured_fp8_source"] = fp8["how"]
    else:
        roof = {"bound": "hbm", "achieved": amount / (kern_ms * 1e-3), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "peak_source": f"{peaks['source']} copy bandwidth (half reads, half writes; a read-only stream can "
                               "exceed it, so frac may pass 1)",
                "frac_vs_nominal_8000": amount / (kern_ms * 1e-3) / 8000.0}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel_ms"] = kern_ms
    roof["kernel"] = {1: "attn_general_kernel", 2: "attn_prefill_kernel", 3: "attn_decode_kernel"}.get(kernel_id, "?")
    roof["traffic"] = ncu_traffic(workload, roof["kernel"])
    return roof


def run_ours(args, rank, world, dev):
    import torch
    import torch.distributed as dist
    from paper_2606_06521_b200 import fp8attn as fa
    cfg_name, kind, mode, S, order = WORKLOADS[args.workload]
    cfg = W.CONFIGS[cfg_name]
    peaks = load_peaks()
    q, k, v, sc = build_device_workload(cfg, kind, seed=rank, dev=dev)
    o = torch.empty((cfg.B, cfg.Hq, cfg.Lq, cfg.d), dtype=torch.float32, device=dev)
    amount, unit, bound = units(cfg, kind)

    def step():
        return fa.fwd(q, k, v, causal=cfg.causal, S=S, kv_order=order, mode=mode, out=o, **sc)

    per_step, total_ms, clocks, r = timed_steps(step, args.steps, args.warmup, dev, world)
    if world > 1:
        dist.barrier()
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms = total_ms / args.steps
    value = world * amount / (ms * 1e-3)

    # ---- end to end: host buffers through fp8attn_fwd_host (H2D + kernels + D2H every step)
    e2e = None
    if rank == 0 or world > 1:
        hq, hk, hv = (t.cpu().pin_memory() for t in (q, k, v))
        hsc = {n: t.cpu() for n, t in sc.items()}
        ho = torch.empty(o.shape, dtype=torch.float32).pin_memory()
        n_e2e = max(1, min(args.steps, 5))

        def estep():
            fa.fwd_host(hq, hk, hv, causal=cfg.causal, S=S, kv_order=order, mode=mode, out=ho, device=dev, **hsc)

        estep()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            estep()                      # synchronises its stream before returning
        el = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([el], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            el = float(t.item())
        h2d = sum(t.numel() * t.element_size() for t in (hq, hk, hv)) + sum(t.numel() * 4 for t in hsc.values())
        e2e = {"value": world * amount / (el / n_e2e), "unit": unit, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(ho.numel() * 4), "steps": n_e2e, "ms_per_step": 1e3 * el / n_e2e,
               "api": "fp8attn_fwd_host (pinned host q,k,v -> o)"}
        assert torch.equal(ho, o.cpu()), "fp8attn_fwd_host and fp8attn_fwd disagree"
        del hq, hk, hv, ho

    # ---- the same launch with statistics on ("separate run with stats on to show its cost"):
    # row_max / row_sum and the two underflow counters from the statistics instance of the prefill kernel
    stats_cost = None
    if bound == "tensor" and rank == 0 and r.kernel_id == 2:
        def sstep():
            return fa.fwd(q, k, v, causal=cfg.causal, S=S, kv_order=order, mode=mode, out=o, kernel=2,
                          want_stats=True, **sc)
        rs = sstep()
        torch.cuda.synchronize()
        n_s = max(1, min(args.steps, 10))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n_s):
            rs = sstep()
        e1.record()
        torch.cuda.synchronize()
        uf = [int(x) for x in rs.underflow.cpu()]
        stats_cost = {"ms_per_step": e0.elapsed_time(e1) / n_s, "steps": n_s, "kernel_id": rs.kernel_id,
                      "underflow_sink_block": uf[0], "underflow_other_blocks": uf[1],
                      "value": amount / (e0.elapsed_time(e1) / n_s * 1e-3), "unit": unit}
        del rs

    kern_ms = float(np.mean(per_step))
    roof = roofline_of(args.workload, cfg, mode, bound, amount, kern_ms, r.kernel_id, peaks)
    line = {
        "metric": "FP8 attention forward throughput" if bound == "tensor" else "split-KV decode attention bandwidth",
        "value": value, "unit": unit, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms, "ms_median": float(np.median(per_step)), "ms_best": float(np.min(per_step)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "e4m3 (fp32 accumulate)" if mode == 2 else "bf16 (fp32 accumulate), P cast to e4m3",
        "data": "synthetic",
        "config": config_of(args.workload, r.block_m, r.block_n, r.num_splits),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(r.n_launches * args.steps),
        "roofline": roof,
    }
    if stats_cost is not None:
        line["with_statistics"] = stats_cost
    del q, k, v, o
    torch.cuda.empty_cache()
    return line


# --------------------------------------------------------------------------- CPU oracle legs
class OracleSample:
    """A bounded sample of the workload for the CPU oracle: whole (b, kv head) slabs are built
    on the host with the same generator, then `n_rows` query rows of one q head are evaluated
    (rows are independent, Alg. 1 is single-row).  Everything here calls only oracle/."""

    def __init__(self, workload, seed=0, kv_head=0, qkv=None):
        import oracle
        self.oracle = oracle
        cfg_name, self.kind, self.mode, self.S, self.order = WORKLOADS[workload]
        self.cfg = cfg = W.CONFIGS[cfg_name]
        q, k, v = W.batch_qkv(cfg, 0, seed) if qkv is None else qkv
        g = cfg.Hq // cfg.Hkv
        self.q = q[None, kv_head * g:(kv_head + 1) * g]       # the q heads of this kv head
        self.k, self.v = k[None, kv_head:kv_head + 1], v[None, kv_head:kv_head + 1]
        _, self.block_n, ns = TILING[workload]
        nb = (cfg.Lk + self.block_n - 1) // self.block_n
        self.split_bounds = [(s * nb) // ns for s in range(ns + 1)] if ns > 1 else None
        if self.kind == "bf16":
            self.q, self.k, self.v = (W.to_bf16_bits(a) for a in (self.q, self.k, self.v))
            self.dt, self.sc = oracle.DT_BF16, {}
        else:
            kc, ks = oracle.quantize_e4m3(self.k)
            vc, vs = oracle.quantize_e4m3(self.v)
            if self.kind == "e4m3":
                qc, qs = oracle.quantize_e4m3(self.q)
                self.q, self.dt = qc, oracle.DT_E4M3
                self.sc = {"q_scale": qs, "k_scale": ks, "v_scale": vs}
            else:
                self.q, self.dt = W.to_bf16_bits(self.q), oracle.DT_BF16Q_E4M3KV
                self.sc = {"k_scale": ks, "v_scale": vs}
            self.k, self.v = kc, vc
        self.n_total = g * cfg.Lq
        self.rng = np.random.default_rng(12345)

    def amount(self, rows):
        """Units of the metric the given rows account for."""
        cfg = self.cfg
        i = rows % cfg.Lq
        vis = np.minimum(cfg.Lk, i + 1 + cfg.Lk - cfg.Lq) if cfg.causal else np.full(len(rows), cfg.Lk)
        if cfg.name == "cfg5":
            # decode: a row re-reads its kv head's K and V (GB of KV per second, per q head)
            return float(np.sum(vis) * cfg.d * 2) / 1e9
        return float(np.sum(vis) * 4.0 * cfg.d) / 1e12

    def run(self, n_rows):
        n_rows = int(min(max(1, n_rows), self.n_total))
        rows = np.sort(self.rng.choice(self.n_total, size=n_rows, replace=False)).astype(np.int64)
        t0 = time.perf_counter()
        res = self.oracle.attention_fwd(self.q, self.k, self.v, causal=self.cfg.causal, S=self.S, kv_order=self.order,
                                        mode=self.mode, in_dtype=self.dt, block_n=self.block_n, rows=rows,
                                        split_bounds=self.split_bounds, **self.sc)
        el = time.perf_counter() - t0
        return self.amount(rows), el, res.n_threads, n_rows

    def rows_for(self, seconds):
        a, el, _, n = self.run(min(64, self.n_total))
        per_row = max(el / n, 1e-6)
        return int(max(8, min(self.n_total, seconds / per_row)))


def cpu_baseline(workload, unit, seconds=12.0):
    """The oracle, as it stands, on a bounded sample: query rows of the q heads of kv head 0, 1, ... of batch
    element 0 until about `seconds` of oracle time have been spent (input preparation is not timed)."""
    cfg = W.CONFIGS[WORKLOADS[workload][0]]
    qkv = W.batch_qkv(cfg, 0, 0)
    amount = el = 0.0
    rows = heads = 0
    threads = 1
    while el < seconds and heads < cfg.Hkv:
        smp = OracleSample(workload, kv_head=heads, qkv=qkv)
        n = smp.rows_for(seconds - el)
        a, t, threads, n = smp.run(n)
        amount, el, rows, heads = amount + a, el + t, rows + n, heads + 1
    return {"value": amount / el, "unit": unit, "cores": threads, "kind": "oracle",
            "sample": f"{rows} random query rows of the q heads of kv heads 0..{heads - 1} of batch element 0 of {workload}, "
                      f"all visible keys; {el:.1f} s of oracle/fp8attn_oracle.c (FP64, OpenMP)"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; a step = a bounded sample."""
    cfg_name, kind, mode, S, order = WORKLOADS[args.workload]
    cfg = W.CONFIGS[cfg_name]
    amount_step, unit, _ = units(cfg, kind)
    smp = OracleSample(args.workload)
    budget = 150.0 / max(1, args.steps + max(args.warmup, 1))
    n = smp.rows_for(min(4.0, budget))
    for _ in range(max(args.warmup, 1)):
        smp.run(n)
    tot_a = tot_t = 0.0
    threads = 1
    for _ in range(args.steps):
        a, el, threads, _ = smp.run(n)
        tot_a += a
        tot_t += el
    value = tot_a / tot_t
    ms = 1e3 * tot_t / args.steps
    return {
        "impl": "reference", "metric": "FP8 attention forward throughput" if unit == "TFLOP/s" else "split-KV decode attention bandwidth",
        "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps, "warmup": max(args.warmup, 1),
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64 (CPU oracle; E4M3 rounding by table)", "data": "synthetic",
        "config": config_of(args.workload, *TILING[args.workload]),
        "cpu_baseline": {"value": value, "unit": unit, "cores": threads, "kind": "oracle",
                         "sample": f"each step = {n} random query rows of (b=0, kv head 0) of {args.workload}, all visible keys"},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# --------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="cfg3")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configs and the CPU baseline")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return 0

    import torch
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the product path has no CPU fallback", file=sys.stderr)
        return 2
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    line = run_ours(args, rank, world, dev)
    if rank == 0 and not args.no_extra and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload, line["unit"])
        # every other BASELINE throughput config beside the headline, each with its own roofline and clock record
        line["extra"] = {}
        for other in ("cfg3", "cfg4-fp8", "cfg4-bf16", "cfg5"):
            if other == args.workload:
                continue
            sub = argparse.Namespace(**{**vars(args), "workload": other, "steps": min(args.steps, 20)})
            try:
                line["extra"][other] = run_ours_extra(sub, dev)
            except Exception as e:      # an extra measurement never takes the headline down
                line["extra"][other] = {"error": repr(e)}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_ours_extra(args, dev):
    """One more workload measured the same way as the headline (device-resident inputs, CUDA events, clocks under
    the same load), without the end-to-end and CPU legs."""
    import torch
    from paper_2606_06521_b200 import fp8attn as fa
    cfg_name, kind, mode, S, order = WORKLOADS[args.workload]
    cfg = W.CONFIGS[cfg_name]
    q, k, v, sc = build_device_workload(cfg, kind, seed=0, dev=dev)
    o = torch.empty((cfg.B, cfg.Hq, cfg.Lq, cfg.d), dtype=torch.float32, device=dev)
    amount, unit, bound = units(cfg, kind)

    def step():
        return fa.fwd(q, k, v, causal=cfg.causal, S=S, kv_order=order, mode=mode, out=o, **sc)

    per_step, total_ms, clocks, r = timed_steps(step, args.steps, 3, dev)
    ms = total_ms / args.steps
    out = {"value": amount / (ms * 1e-3), "unit": unit, "ms_per_step": ms, "ms_median": float(np.median(per_step)),
           "ms_best": float(np.min(per_step)), "steps": args.steps, "kernel_id": r.kernel_id,
           "num_splits": r.num_splits, "block_n": r.block_n, "gpu_launches_per_step": r.n_launches,
           "dtype": "e4m3 (fp32 accumulate)" if mode == 2 else "bf16 (fp32 accumulate), P cast to e4m3",
           "config": config_of(args.workload, r.block_m, r.block_n, r.num_splits),
           "clocks": clocks,
           "roofline": roofline_of(args.workload, cfg, mode, bound, amount, float(np.mean(per_step)), r.kernel_id,
                                   load_peaks())}
    if cfg.name == "cfg5":
        # the same launch with the statistics instance of the decode kernel (P dump off, both underflow counters on)
        def sstep():
            return fa.fwd(q, k, v, causal=cfg.causal, S=S, kv_order=order, mode=mode, out=o, want_stats=True, **sc)
        rs = sstep()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(10):
            rs = sstep()
        e1.record()
        torch.cuda.synchronize()
        uf = [int(x) for x in rs.underflow.cpu()]
        out["with_statistics"] = {"ms_per_step": e0.elapsed_time(e1) / 10, "kernel_id": rs.kernel_id,
                                  "value": amount / (e0.elapsed_time(e1) / 10 * 1e-3), "unit": unit,
                                  "underflow_sink_block": uf[0], "underflow_other_blocks": uf[1]}
    del q, k, v, o
    torch.cuda.empty_cache()
    return out


if __name__ == "__main__":
    sys.exit(main())
