#!/usr/bin/env python
"""bench.py — split-MLP forward+backward throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--k 4] [--graph] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (steps A0-A8: osdp_split_mlp_forward then osdp_split_mlp_backward
through the C ABI) over one batch of seeded synthetic input of the named workload.  `value` is executed
TFLOP/s (14 T h f per step: 4 forward + 8 backward + 2 for the slice recompute of Z the method itself needs),
summed over ranks (each rank runs the operator on its own token batch: data parallelism, weak scaling, no
data-path collective).  Inputs are resident in HBM for `value`; `e2e` is the same metric with host (pinned)
buffers, host<->device copies of every input and output inside the timed region (three streams, so the copies
of neighbouring steps overlap the kernels; the unpipelined figure is reported beside it).

`--impl reference` times the fp64 CPU oracle (oracle/mlp_oracle.py) as it stands on the box's host cores on a
bounded token sample of the same workload (the reference arm of this tier); only rank 0 runs it.
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

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

METRIC = "split_mlp_fwd_bwd_tflops"
UNIT = "TFLOP/s"
NOMINAL_BF16_TFLOPS = 2250.0      # dense bf16, B200 (B200_PROFILING.md; context only)
# GEMMs (of 2 T_s h f flops each) per traced launch: steps A1-A7 are one GEMM; the one-kernel-per-slice launches (small
# slices, csrc/slice_sm100.cuh) hold the forward's two (step 21) / the backward's five (step 22)
GEMMS_PER_LAUNCH = {1: 1, 2: 1, 3: 1, 4: 1, 5: 1, 6: 1, 7: 1, 21: 2, 22: 5}
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
L2_BYTES = 126 << 20


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        d["source"] = "measured"
        return d
    d = dict(FALLBACK_PEAKS)
    d["source"] = "fallback"
    return d


def executed_flops(T, h, f):
    return 14.0 * T * h * f


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe): NVML polled
    every 20 ms from a thread (the timed region of a default run is a few hundred ms, too short for nvidia-smi's
    start-up); `nvidia-smi -lms 100` is the fallback when NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.proc, self.thread, self.running = index, None, None, False
        self.lines, self.samples, self.reasons, self.max_mhz = [], [], set(), None
        self.nv = self.handle = None
        try:
            import pynvml
            pynvml.nvmlInit()
            dev = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = int(dev.split(",")[index]) if dev and all(x.strip().isdigit() for x in dev.split(",")) else index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nv = pynvml
        except Exception:
            self.nv = None

    def _poll_nvml(self):
        nv = self.nv
        bits = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(nv, "nvmlDeviceGetCurrentClocksThrottleReasons")
        while self.running:
            try:
                self.samples.append((float(nv.nvmlDeviceGetClockInfo(self.handle, nv.NVML_CLOCK_SM)),
                                     nv.nvmlDeviceGetPowerUsage(self.handle) / 1e3))
                r = int(get_reasons(self.handle))
                for nm, bit in bits.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.02)

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def start(self):
        if self.nv is not None:
            self.running = True
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def stop(self):
        if self.nv is not None:
            self.running = False
            self.thread.join()
            sm = [x[0] for x in self.samples]
            pw = [x[1] for x in self.samples]
            return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": self.max_mhz,
                    "power_w_max": max(pw) if pw else None, "reasons": sorted(self.reasons), "samples": len(sm),
                    "source": "nvml, 20 ms"}
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "source": "none"}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(self.NAMES, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm),
                "source": "nvidia-smi -lms 100"}


def barrier(world):
    from paper_2305_09940_b200 import dist as D
    D.barrier()


def max_over_ranks(x, world):
    from paper_2305_09940_b200 import dist as D
    return D.max_over_ranks(x)


# --------------------------------------------------------------------------------------------- reference arm
def oracle_sample_tokens(h, f, target_flops=2.5e12):
    """Token sample for the CPU oracle: about 10-30 s of fp64 work on a few dozen cores."""
    t = int(target_flops / (14.0 * h * f))
    return max(8, min(4096, 1 << max(0, t.bit_length() - 1)))


def time_oracle(cfg, steps, warmup, sample_tokens=None):
    """Times oracle.mlp_forward_backward as it stands on the first T' tokens of the workload."""
    import numpy as np  # noqa: F401
    from oracle import mlp_oracle as O
    from paper_2305_09940_b200 import inputs as I
    T, h, f = cfg["tokens"], cfg["hidden"], cfg["ffn"]
    Ts = sample_tokens or oracle_sample_tokens(h, f)
    Ts = min(Ts, T)
    dt = I.torch_dtype(cfg["dtype"])
    t0 = time.time()
    inp = I.mlp_inputs(Ts, h, f, dt, seed=cfg["seed"])
    x = inp.as_f64()
    log(f"[oracle] inputs for T'={Ts} tokens generated in {time.time() - t0:.1f}s")
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        O.mlp_forward_backward(**x)
        dtm = time.perf_counter() - t0
        if i >= warmup:
            times.append(dtm)
    sec = sum(times) / len(times)
    cores = os.cpu_count() or 1
    try:
        import threadpoolctl
        infos = [i for i in threadpoolctl.threadpool_info() if i.get("user_api") == "blas"]
        if infos:
            cores = max(i["num_threads"] for i in infos)
    except Exception:
        pass
    return {"value": executed_flops(Ts, h, f) / sec / 1e12, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": f"first {Ts} of {T} tokens, full hidden={h} ffn={f}, fp64 numpy; cost is linear in tokens",
            "seconds_per_sample": sec, "sample_tokens": Ts}


def run_reference(args, cfg, rank):
    if rank != 0:
        return
    r = time_oracle(cfg, max(1, min(args.steps, 3)), min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": max(1, min(args.steps, 3)), "warmup": min(args.warmup, 1),
            "ms_per_step": r["seconds_per_sample"] * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, cfg), "tokens": cfg["tokens"], "hidden": cfg["hidden"],
                       "ffn": cfg["ffn"], "k": args.k, "sample_tokens": r["sample_tokens"]},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_name(args, cfg):
    return (f"{args.config}: MLP operator tokens={cfg['tokens']} hidden={cfg['hidden']} ffn={cfg['ffn']} "
            f"{cfg['dtype']}, fwd+bwd at k={args.k} {'token' if args.axis == 'tokens' else 'ffn'} slices")


# --------------------------------------------------------------------------------------------------- our arm
class Workload:
    def __init__(self, lib, cfg, k, seed):
        from paper_2305_09940_b200 import inputs as I
        self.lib = lib
        self.T, self.h, self.f = cfg["tokens"], cfg["hidden"], cfg["ffn"]
        self.dtype = I.torch_dtype(cfg["dtype"])
        t0 = time.time()
        self.host = I.mlp_inputs(self.T, self.h, self.f, self.dtype, seed=seed, pin=True)
        log(f"[bench] seeded host inputs generated in {time.time() - t0:.1f}s")
        self.dev = self.host.to("cuda")
        e = torch.empty
        self.Y = e((self.T, self.h), dtype=self.dtype, device="cuda")
        self.g = dict(dX=e((self.T, self.h), dtype=self.dtype, device="cuda"),
                      dW1=e((self.h, self.f), dtype=torch.float32, device="cuda"),
                      db1=e((self.f,), dtype=torch.float32, device="cuda"),
                      dW2=e((self.f, self.h), dtype=torch.float32, device="cuda"),
                      db2=e((self.h,), dtype=torch.float32, device="cuda"))
        self.set_k(k)
        # host-side result buffers for the e2e leg
        self.hY = e((self.T, self.h), dtype=self.dtype, pin_memory=True)
        self.hg = {n: e(t.shape, dtype=t.dtype, pin_memory=True) for n, t in self.g.items()}

    def set_k(self, k, axis="tokens"):
        self.k, self.axis = k, axis
        self.op = None
        torch.cuda.empty_cache()
        self.op = self.lib.SplitMlp(self.T, self.h, self.f, self.dtype, k, axis=axis)

    def step(self):
        d = self.dev
        self.op.forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=self.Y)
        n = self.lib.osdp_last_launch_count()
        self.op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=self.g)
        return n + self.lib.osdp_last_launch_count()

    def step_e2e(self):
        """Host buffers in, host buffers out: H2D of every input, the path, D2H of every output."""
        h, d = self.host, self.dev
        for n in ("X", "W1", "b1", "W2", "b2", "dY"):
            getattr(d, n).copy_(getattr(h, n), non_blocking=True)
        self.step()
        self.hY.copy_(self.Y, non_blocking=True)
        for n, t in self.g.items():
            self.hg[n].copy_(t, non_blocking=True)

    def run_e2e_pipelined(self, steps, world):
        """The same per-step work as step_e2e (H2D of every input from pinned host memory, forward + backward, D2H of
        every output), as a user's input pipeline would run it: three streams, device tensors double-buffered, so the
        H2D of step i+1 and the D2H of step i-1 overlap the kernels of step i (PCIe is full duplex).  Returns ms/step
        measured with CUDA events around all `steps` steps, barrier + synchronize on both sides."""
        e = torch.empty
        names = ("X", "W1", "b1", "W2", "b2", "dY")
        ins = [self.dev, self.host.to("cuda")]
        outs = [(self.Y, self.g), (torch.empty_like(self.Y), {n: torch.empty_like(t) for n, t in self.g.items()})]
        s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
        ev_in = [torch.cuda.Event() for _ in range(2)]      # inputs of set b uploaded
        ev_cmp = [torch.cuda.Event() for _ in range(2)]     # kernels that read set b / wrote out set b finished
        ev_out = [torch.cuda.Event() for _ in range(2)]     # outputs of set b read back
        start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def run(n, timed):
            cur = torch.cuda.current_stream()
            for st in (s_in, s_cmp, s_out):
                st.wait_stream(cur)
            if timed:
                start.record(cur)
                for st in (s_in, s_cmp, s_out):
                    st.wait_event(start)
            for i in range(n):
                b = i % 2
                with torch.cuda.stream(s_in):
                    if i >= 2:
                        s_in.wait_event(ev_cmp[b])          # the kernels of step i-2 no longer read this input set
                    for nm in names:
                        getattr(ins[b], nm).copy_(getattr(self.host, nm), non_blocking=True)
                    ev_in[b].record(s_in)
                with torch.cuda.stream(s_cmp):
                    s_cmp.wait_event(ev_in[b])
                    if i >= 2:
                        s_cmp.wait_event(ev_out[b])         # the outputs of step i-2 have been read back
                    Y, g = outs[b]
                    d = ins[b]
                    self.op.forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=Y, stream=s_cmp)
                    self.op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=g, stream=s_cmp)
                    ev_cmp[b].record(s_cmp)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_cmp[b])
                    Y, g = outs[b]
                    self.hY.copy_(Y, non_blocking=True)
                    for nm, t in g.items():
                        self.hg[nm].copy_(t, non_blocking=True)
                    ev_out[b].record(s_out)
            for st in (s_in, s_cmp, s_out):
                cur.wait_stream(st)
            if timed:
                stop.record(cur)

        run(3, False)
        barrier(world)
        run(steps, True)
        barrier(world)
        return start.elapsed_time(stop) / steps

    def h2d_bytes(self):
        return sum(getattr(self.host, n).numel() * getattr(self.host, n).element_size()
                   for n in ("X", "W1", "b1", "W2", "b2", "dY"))

    def d2h_bytes(self):
        return self.hY.numel() * self.hY.element_size() + sum(t.numel() * t.element_size() for t in self.hg.values())

    def resident_bytes(self):
        return self.h2d_bytes() + self.d2h_bytes()


def timed_steps(fn, steps, world, flush=None):
    """EXACTLY `steps` steps between barrier+synchronize brackets; per-step CUDA events on the current stream.
    Returns (sum of step ms, wall ms of the bracket); the per-step times of the last call are kept in
    timed_steps.last (median and min are reported beside the mean)."""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier(world)
    t0 = time.perf_counter()
    for a, b in evs:
        if flush is not None:
            flush.zero_()
        a.record()
        fn()
        b.record()
    barrier(world)
    wall = (time.perf_counter() - t0) * 1e3
    timed_steps.last = [a.elapsed_time(b) for a, b in evs]
    return sum(timed_steps.last), wall


timed_steps.last = []


def graph_step_ms(wl, steps, world, flush):
    """The same step captured once in a CUDA graph and replayed: what is left of the host-side launch cost (tensor-map
    encoding, argument checks, ~10 launches per slice) disappears; the kernels are the same.  Returns ms/step."""
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for _ in range(2):
            wl.step()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        wl.step()
    for _ in range(3):
        g.replay()
    ms, _ = timed_steps(g.replay, steps, world, flush)
    return ms / steps, statistics.median(timed_steps.last), min(timed_steps.last)


def measure_peak_bytes(lib, cfg, k, axis="tokens"):
    """Peak device bytes of ONE forward call and ONE backward call, each with only its own tensors live,
    against the cost model (osdp_mlp_op_cost + osdp_cost_eval)."""
    from paper_2305_09940_b200 import inputs as I
    T, h, f = cfg["tokens"], cfg["hidden"], cfg["ffn"]
    dt = I.torch_dtype(cfg["dtype"])
    out = {}
    for name, pass_ in (("fwd", lib.OSDP_FWD), ("bwd", lib.OSDP_BWD)):
        torch.cuda.synchronize()
        torch.cuda.empty_cache()
        base = torch.cuda.memory_allocated()
        free0, _ = torch.cuda.mem_get_info()            # the device's own view (cudaMemGetInfo), not the allocator's
        torch.cuda.reset_peak_memory_stats()
        desc = lib.make_desc(T, h, f, dt, k)
        mk = lambda *s, d=dt: torch.empty(s, dtype=d, device="cuda")
        X, W1, b1, W2, b2 = mk(T, h), mk(h, f), mk(f), mk(f, h), mk(h)
        ffn = axis == "ffn"
        ws_bytes = (lib.osdp_ffn_split_mlp_workspace_bytes if ffn else lib.osdp_split_mlp_workspace_bytes)(desc, pass_)
        ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
        for t in (X, W1, b1, W2, b2):
            t.zero_()
        if pass_ == lib.OSDP_FWD:
            Y = mk(T, h)
            (lib.osdp_ffn_split_mlp_forward if ffn else lib.osdp_split_mlp_forward)(desc, X, W1, b1, W2, b2, Y, ws)
        else:
            dY, dX = mk(T, h), mk(T, h)
            dY.zero_()
            f32 = torch.float32
            dW1, db1, dW2, db2 = mk(h, f, d=f32), mk(f, d=f32), mk(f, h, d=f32), mk(h, d=f32)
            (lib.osdp_ffn_split_mlp_backward if ffn else lib.osdp_split_mlp_backward)(
                desc, X, W1, b1, W2, b2, dY, dX, dW1, db1, dW2, db2, ws)
        torch.cuda.synchronize()
        measured = torch.cuda.max_memory_allocated() - base
        free1, _ = torch.cuda.mem_get_info()            # all call tensors still alive here: used-memory delta of the device
        c = (lib.osdp_ffn_split_mlp_op_cost if ffn else lib.osdp_mlp_op_cost)(desc, pass_)
        dev = lib.osdp_device(1, 0.0, 0.0, 1 << 62)
        p, tr, _ = lib.osdp_cost_eval(c, lib.OSDP_DP, k, 1, dev)
        model = int(p + tr)
        if ffn and k == 1:       # the variant's cost factors describe k > 1; at k = 1 there is no fp32 accumulator
            model -= (T * h * 4 + 255) // 256 * 256
        out[name] = {"measured": int(measured), "model": model, "workspace": int(ws.numel()),
                     "device_used_delta": int(free0 - free1)}   # >= measured by the allocator's 2 MiB segment rounding; the library allocates nothing itself
        del X, W1, b1, W2, b2, ws
        if pass_ == lib.OSDP_FWD:
            del Y
        else:
            del dY, dX, dW1, db1, dW2, db2
    torch.cuda.empty_cache()
    return out


def other_configs_table(lib, peaks, local_gpu, steps=10):
    """BASELINE.json's other single-operator configurations, timed in the same run as the headline line so that their
    figures are the driver's, not only the builder's: C1 (fp32) k = 4, C2 k in {1, 4, 8}, C3 k = 4 and the operator of one
    C5 layer at k = 4 (the 24-layer stack itself stays under --config C5 --stack).  Inputs are RESIDENT and generated on
    the device (seeded torch.randn with the recipe's distributions: X, dY ~ N(0, 1), W, b ~ N(0, 0.02)) - parity on the
    seeded host inputs is the tests' job; here only time is measured.  Each row: forward + backward through the C ABI,
    3 warm-up + `steps` timed steps with per-step CUDA events, a 256 MiB memset between steps when the tensors fit L2.
    frac = TFLOP/s over the measured sustained bf16 peak (bf16) or over the FFMA peak at the SM clock sampled while the
    table ran (fp32)."""
    from paper_2305_09940_b200 import inputs as I
    rows = []
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    sampler = ClockSampler(local_gpu)
    sampler.start()
    for name, k in (("C1", 4), ("C2", 1), ("C2", 4), ("C2", 8), ("C3", 4), ("C5", 4)):
        c = I.CONFIGS[name]
        T, h, f, dt = c["tokens"], c["hidden"], c["ffn"], I.torch_dtype(c["dtype"])
        gen = torch.Generator(device="cuda").manual_seed(c["seed"])
        rn = lambda *shape, std=1.0: (torch.randn(*shape, device="cuda", generator=gen) * std).to(dt)
        X, dY = rn(T, h), rn(T, h)
        W1, b1, W2, b2 = rn(h, f, std=0.02), rn(f, std=0.02), rn(f, h, std=0.02), rn(h, std=0.02)
        Y = torch.empty_like(X)
        g = dict(dX=torch.empty_like(X), dW1=torch.empty(h, f, device="cuda"), db1=torch.empty(f, device="cuda"),
                 dW2=torch.empty(f, h, device="cuda"), db2=torch.empty(h, device="cuda"))
        op = lib.SplitMlp(T, h, f, dt, k)
        launches = [0]

        def step():
            op.forward(X, W1, b1, W2, b2, Y=Y)
            n = lib.osdp_last_launch_count()
            op.backward(X, W1, b1, W2, dY, out=g)
            launches[0] = n + lib.osdp_last_launch_count()

        for _ in range(3):
            step()
        resident = sum(t.numel() * t.element_size() for t in (X, dY, W1, b1, W2, b2, Y, *g.values()))
        small = resident < 2 * L2_BYTES
        ms_sum, _ = timed_steps(step, steps, 1, flush if small else None)
        ms = ms_sum / steps
        rows.append({"config": name + (" (one layer's operator)" if name == "C5" else ""), "tokens": T, "hidden": h, "ffn": f,
                     "dtype": c["dtype"], "k": k, "ms_per_step": ms, "ms_per_step_min": min(timed_steps.last),
                     "tflops": executed_flops(T, h, f) / (ms * 1e-3) / 1e12, "gpu_launches_per_step": int(launches[0]),
                     "l2": "flush between steps" if small else "tensors exceed L2"})
        del op, X, dY, W1, b1, W2, b2, Y, g
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    bf16_peak = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    ghz = (clocks.get("sm_mhz") or 1965.0) * 1e-3
    for r in rows:
        if r["dtype"] == "bf16":
            r["frac"], r["frac_of"] = r["tflops"] / bf16_peak, "measured sustained bf16 peak (step level)"
        else:
            r["frac"] = r["tflops"] / (148 * 128 * 2 * ghz * 1e-3)
            r["frac_of"] = f"FFMA peak 148 SMs x 128 x 2 x {ghz:.3f} GHz (clock sampled while the table ran)"
    return {"rows": rows, "clocks": clocks, "data": "resident, generated on the device (seeded torch.randn, the recipe's distributions)",
            "steps": steps, "warmup": 3}


def fit_gamma_delta(table):
    """Device information for the planner ("profiled in advance"), from the per-k sweep: the cost model's
    T(k) = gamma + (k - 1) delta (reading P2) with gamma = the measured k = 1 time and delta the least-squares
    slope through it; max_rel_residual says how well the linear model holds."""
    t1 = next((e["ms_per_step"] for e in table if e["k"] == 1), None)
    pts = [(e["k"] - 1, e["ms_per_step"] - t1) for e in table if e["k"] > 1] if t1 is not None else []
    if not pts:
        return None
    delta = sum(x * y for x, y in pts) / sum(x * x for x, _ in pts)
    resid = max(abs(t1 + x * delta - (t1 + y)) / (t1 + y) for x, y in pts)
    return {"gamma_s": t1 * 1e-3, "delta_s": delta * 1e-3, "max_rel_residual": resid}


def granularity_sweep(args, lib):
    """Time and peak device bytes against the slice granularity for small and large operators ("for
    models with small hidden sizes the time cost increases as the slice granularity gets larger", large operators
    "require larger slice granularity" for the memory benefit).  The paper sweeps granularity 0-16 with hidden 768 /
    1024 and 8192 / 12288 under ZDP on 8 GPUs; here: one GPU, one MLP operator, both split axes, k = 1 (the paper's
    0) to 16.  One JSON line."""
    rows = []
    ks = (1, 2, 4, 8, 16)
    for h in [int(x) for x in args.granularity_sweep.split(",")]:
        cfg = dict(tokens=args.sweep_tokens, hidden=h, ffn=4 * h, dtype="bf16", seed=0)
        wl = Workload(lib, cfg, 1, seed=0)
        flops = executed_flops(cfg["tokens"], h, 4 * h)
        small = wl.resident_bytes() < 2 * L2_BYTES
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None
        for axis in ("tokens", "ffn"):
            for k in ks:
                wl.set_k(k, axis)
                for _ in range(3):
                    wl.step()
                torch.cuda.synchronize()
                n = max(5, min(200, int(0.5 / max(1e-5, flops / 1.2e15))))     # about half a second per point
                ms, _ = timed_steps(wl.step, n, 1, flush)
                rows.append({"hidden": h, "axis": axis, "k": k, "steps": n, "ms_per_step": ms / n,
                             "tflops": flops / (ms / n * 1e-3) / 1e12})
        del wl, flush
        torch.cuda.empty_cache()
        for r in rows:
            if r["hidden"] == h:
                pk = measure_peak_bytes(lib, cfg, r["k"], r["axis"])
                r["peak_bytes_fwd"], r["peak_bytes_bwd"] = pk["fwd"]["measured"], pk["bwd"]["measured"]
                r["model_bytes_fwd"], r["model_bytes_bwd"] = pk["fwd"]["model"], pk["bwd"]["model"]
    print(json.dumps({"granularity_sweep": rows, "tokens": args.sweep_tokens, "unit": UNIT, "dtype": "bf16",
                      "data": "synthetic", "cite": "PAPER.md:231-247 (Fig. 7): shape only, the figure's numbers are an image"}),
          flush=True)
    return 0


def stack_bench(args, lib, cfg):
    """BASELINE.json config 5: a chain of `layers` MLP operators (X_{l+1} = MLP_l(X_l), reading S13), forward through
    all layers then backward, the split count of each layer chosen by osdp_plan under the activation cap.
    Device information for the planner (alpha, beta, gamma "profiled in advance") is calibrated here:
    one layer is timed at k = 1, 2, 4, 8, 16 and T(k) = gamma + (k - 1) delta is fitted (fit_gamma_delta).  The
    memory factors are the paper's accounting (Eq. 1 sums M_i over operators; 8 B per T x f element for an unfused
    autograd MLP, SURVEY.md section 8 note), under which the 24 GiB cap binds.  One JSON line: measured stack
    throughput, the plan, and the planner's time estimate next to the measured time."""
    from paper_2305_09940_b200 import inputs as I
    T, h, f, L = cfg["tokens"], cfg["hidden"], cfg["ffn"], cfg.get("layers", 24)
    dt = I.torch_dtype(cfg["dtype"])
    ks_cal = (1, 2, 4, 8, 16)
    wl = Workload(lib, cfg, 1, seed=0)
    table = []
    for k in ks_cal:
        wl.set_k(k)
        for _ in range(3):
            wl.step()
        ms, _ = timed_steps(wl.step, 20, 1, None)
        n = max(20, min(400, int(600.0 / max(ms / 20, 1e-3))))      # ~0.6 s per point: at the power cap, like the stack itself
        ms, _ = timed_steps(wl.step, n, 1, None)
        table.append({"k": k, "ms_per_step": ms / n, "steps": n})
    fit = fit_gamma_delta(table)
    del wl
    torch.cuda.empty_cache()

    desc1 = lib.make_desc(T, h, f, dt, 1)
    ops = []
    for _ in range(L):
        oc = lib.osdp_mlp_op_cost(desc1, lib.OSDP_BWD)
        oc.model_bytes = (2 * h * f + f + h) * 2          # weights; gradients / optimizer states outside the activation cap
        oc.extra_fixed = 0
        oc.extra_transient = 0
        oc.extra_summed = 8 * T * f                       # Z, H, dH, dZ in bf16: the unfused-autograd view of the intermediate
        oc.act_bytes = T * h * 2                          # saved layer input
        oc.gamma, oc.delta = fit["gamma_s"], max(fit["delta_s"], 0.0)
        ops.append(oc)
    cap = cfg.get("act_cap_bytes", 24 << 30)
    st, ks, modes, est_s, est_peak = lib.osdp_plan(ops, lib.osdp_device(1, 0.0, 0.0, cap), 1, [1, 2, 4, 8, 16, 32])
    if st != lib.OSDP_OK:
        raise SystemExit(f"osdp_plan: status {st}")

    # ---- memory as the library really uses it (not the paper's accounting above): model states + the T x h tensors
    # the chain keeps per layer (saved input X_l and dX_l; dY_l is dX_{l+1}) summed over layers, ONE transient workspace
    # shared by all layers (slices and layers run one after another: "released serially"), predicted with
    # osdp_mlp_op_cost + osdp_cost_eval for the plan that is run, and measured below as the allocator's peak and as the
    # device's own used-memory delta (cudaMemGetInfo).
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    alloc0 = torch.cuda.memory_allocated()
    torch.cuda.reset_peak_memory_stats()
    real_persist, real_transient = 0, 0
    for l in range(L):
        oc = lib.osdp_mlp_op_cost(desc1, lib.OSDP_BWD)
        oc.act_bytes = 2 * T * h * 2                       # X_l and dX_l
        p_, t_, _ = lib.osdp_cost_eval(oc, lib.OSDP_DP, ks[l], 1, lib.osdp_device(1, 0.0, 0.0, 1 << 62))
        real_persist += p_ - oc.extra_fixed                # the column-sum scratch lives inside the shared workspace
        real_transient = max(real_transient, t_ + oc.extra_fixed)
    est_real = real_persist + real_transient + 2 * T * h * 2        # + X_L (the stack's output) and dY_L

    t0 = time.time()
    layers = []
    ws_bytes = 0
    for l in range(L):
        w = I.mlp_inputs(1, h, f, dt, seed=l)             # weights and biases of layer l (seed = layer, reading S13)
        op = lib.SplitMlp(T, h, f, dt, ks[l])
        ws_bytes = max(ws_bytes, op.workspace.numel())
        op.workspace = None
        layers.append(dict(W1=w.W1.cuda(), b1=w.b1.cuda(), W2=w.W2.cuda(), b2=w.b2.cuda(), op=op,
                           g=dict(dX=torch.empty((T, h), dtype=dt, device="cuda"),
                                  dW1=torch.empty((h, f), dtype=torch.float32, device="cuda"),
                                  db1=torch.empty((f,), dtype=torch.float32, device="cuda"),
                                  dW2=torch.empty((f, h), dtype=torch.float32, device="cuda"),
                                  db2=torch.empty((h,), dtype=torch.float32, device="cuda"))))
    torch.cuda.empty_cache()
    shared_ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")      # one transient workspace for the whole stack
    for ly in layers:
        ly["op"].workspace = shared_ws
    Xs = [I.normal_tensor(0, I.STREAM_X, (T, h), 1.0, dt).cuda()] + [torch.empty((T, h), dtype=dt, device="cuda") for _ in range(L)]
    dYL = I.normal_tensor(0, I.STREAM_DY, (T, h), 1.0, dt).cuda()
    log(f"[bench] stack inputs generated in {time.time() - t0:.1f}s; plan k = {ks}")
    launches = [0]

    def step():
        n = 0
        for l, ly in enumerate(layers):
            ly["op"].forward(Xs[l], ly["W1"], ly["b1"], ly["W2"], ly["b2"], Y=Xs[l + 1])
            n += lib.osdp_last_launch_count()
        dY = dYL
        for l in reversed(range(L)):
            ly = layers[l]
            ly["op"].backward(Xs[l], ly["W1"], ly["b1"], ly["W2"], dY, out=ly["g"])
            n += lib.osdp_last_launch_count()
            dY = ly["g"]["dX"]
        launches[0] = n

    for _ in range(max(3, args.warmup)):
        step()
    steps = max(3, min(args.steps, 20))
    sampler = ClockSampler(0)
    sampler.start()
    ms_sum, _ = timed_steps(step, steps, 1, None)
    clocks = sampler.stop()
    ms = ms_sum / steps
    flops = executed_flops(T, h, f) * L
    peaks = load_peaks()
    torch.cuda.synchronize()
    measured_alloc = torch.cuda.max_memory_allocated() - alloc0
    free1, _ = torch.cuda.mem_get_info()
    memory = {"est_peak_bytes_library_factors": int(est_real), "measured_peak_bytes_allocator": int(measured_alloc),
              "measured_device_used_delta_bytes": int(free0 - free1), "measured_over_est": measured_alloc / est_real,
              "workspace_bytes_shared": int(ws_bytes),
              "note": "library factors: osdp_mlp_op_cost + osdp_cost_eval per layer (model states, X_l, dX_l) + one shared "
                      "transient workspace; the 24 GiB cap does not bind under them (the fused, recomputing path keeps no "
                      "T x f tensor per layer) - est_peak_bytes_paper_accounting is the paper-style sum the cap is meant for"}
    print(json.dumps({
        "metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": cfg["dtype"], "data": "synthetic",
        "config": {"workload": f"C5: {L}-layer MLP stack tokens={T} hidden={h} ffn={f} bf16, fwd through all layers then bwd, "
                               f"k per layer from osdp_plan under a {cap >> 30} GiB activation cap",
                   "k_per_layer": ks, "flops_per_step": flops, "l2": "inputs+outputs exceed L2 (126 MB); no flush"},
        "frac_of_sustained_peak": flops / (ms * 1e-3) / 1e12 / peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]),
        "frac_of_nominal_peak": flops / (ms * 1e-3) / 1e12 / NOMINAL_BF16_TFLOPS,
        "planner": {"calibration_ms_per_layer": {str(e["k"]): e["ms_per_step"] for e in table}, "fit": fit,
                    "est_ms_per_step": est_s * 1e3, "measured_ms_per_step": ms, "est_over_measured": est_s * 1e3 / ms,
                    "est_peak_bytes_paper_accounting": est_peak, "cap_bytes": cap},
        "memory": memory, "clocks": clocks, "gpu_launches": launches[0] * steps}), flush=True)
    return 0


def zdp_bench(args, lib, cfg):
    """ZDP mode with weight-slice gathering: every rank owns its token batch
    and 1/N of the model states; each step = osdp_zdp_ffn_split_mlp_forward + backward with the slice all-gathers and
    reduce-scatters (NCCL through torch.distributed) on a second stream beside the GEMMs.  Works at N = 1 (single-rank
    NCCL group: the collectives are real but move nothing between GPUs); N > 1 has never been run (one-GPU lease).
    One JSON line; `value` = executed TFLOP/s summed over ranks, max-over-ranks device time."""
    import torch.distributed as dist
    from paper_2305_09940_b200 import dist as D
    from paper_2305_09940_b200 import inputs as I
    world, rank, local = D.init("nccl")
    if not dist.is_initialized():        # single process: a one-rank group so that the collectives are real NCCL calls
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29517")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    T, h, f, k = cfg["tokens"], cfg["hidden"], cfg["ffn"], args.zdp
    dt = I.torch_dtype(cfg["dtype"])
    whole = I.mlp_inputs(1, h, f, dt, seed=cfg["seed"])                  # the same weights on every rank
    mine = I.mlp_inputs(T, h, 8, dt, seed=D.rank_seed(cfg["seed"], rank) + 1000)   # this rank's tokens (X, dY)
    desc = lib.make_zdp_desc(T, h, f, dt, k, world, rank)
    shard = lib.zdp_shard(desc, whole.W1, whole.b1, whole.W2, whole.b2).cuda()
    X, dY = mine.X.cuda(), mine.dY.cuda()
    Y, dX = torch.empty_like(X), torch.empty_like(X)
    gshard = torch.empty(shard.numel(), dtype=torch.float32, device="cuda")
    ws = torch.empty(max(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, p) for p in (lib.OSDP_FWD, lib.OSDP_BWD)),
                     dtype=torch.uint8, device="cuda")
    comm, cs = lib.TorchDistComm(), torch.cuda.Stream()
    launches = [0]

    def step():
        lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, X, Y, ws, comm=comm, comm_stream=cs)
        n = lib.osdp_last_launch_count()
        lib.osdp_zdp_ffn_split_mlp_backward(desc, shard, X, dY, dX, gshard, ws, comm=comm, comm_stream=cs)
        launches[0] = n + lib.osdp_last_launch_count()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(local)
    sampler.start()
    ms_sum, _ = timed_steps(step, args.steps, world, None)
    clocks = sampler.stop()
    ms = max_over_ranks(ms_sum / args.steps, world)
    flops = executed_flops(T, h, f)
    e = 2 if cfg["dtype"] == "bf16" else 4
    S = (2 * h * f + f + h) * e
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": world * flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": cfg["dtype"], "data": "synthetic",
            "config": {"workload": f"{args.config}: ZDP ffn-split MLP tokens/GPU={T} hidden={h} ffn={f}, k={k} ffn slices, "
                                   f"model states sharded over {world} ranks, slice gathers / reduce-scatters on a second stream",
                       "parallelism": f"zdp{world}", "collective_bytes_per_rank_per_step":
                           {"all_gather_contributed": (2 * S - h * e) // world, "reduce_scatter_contributed": (S // e) * 4 // world},
                       "workspace_bytes": int(ws.numel()), "param_shard_bytes": int(shard.numel() * e)},
            "clocks": clocks, "gpu_launches": launches[0] * args.steps,
            "note": "N > 1 has not been run on hardware by the builder (one-GPU lease); at N = 1 the NCCL collectives are "
                    "single-rank copies"}), flush=True)
    D.finalize()
    return 0


def vendor_dw_bench(args, cfg):
    """cuBLAS on the dW GEMM shapes (A5: [f x T_s] x [T_s x h], A6: [h x T_s] x [T_s x f]; bf16 operands, fp32 output,
    beta = 0 and beta = 1), each timed in a ~2 s back-to-back loop.  A library reference for the dominant kernel's shape,
    not part of the product path."""
    T, h, f = cfg["tokens"], cfg["hidden"], cfg["ffn"]
    ts = (T + args.k - 1) // args.k
    peaks = load_peaks()

    def sustained(fn, secs=2.0):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(10):
            fn()
        e1.record()
        torch.cuda.synchronize()
        n = max(10, int(secs * 1e3 / (e0.elapsed_time(e1) / 10)))
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n

    rows = []
    for name, (m, n) in (("A5 dW2 = H_s^T dY_s", (f, h)), ("A6 dW1 = X_s^T dZ_s", (h, f))):
        a = torch.randn(ts, m, device="cuda", dtype=torch.bfloat16)
        b = torch.randn(ts, n, device="cuda", dtype=torch.bfloat16)
        c = torch.zeros(m, n, device="cuda", dtype=torch.float32)
        flops = 2.0 * m * n * ts
        ms0 = sustained(lambda: torch.mm(a.t(), b, out_dtype=torch.float32, out=c))
        ms1 = sustained(lambda: torch.addmm(c, a.t(), b, out_dtype=torch.float32, out=c))
        rows.append({"gemm": name, "M": m, "N": n, "K": ts, "beta0_ms": ms0, "beta0_tflops": flops / ms0 / 1e9,
                     "beta1_ms": ms1, "beta1_tflops": flops / ms1 / 1e9})
        del a, b, c
    sus = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"])
    print(json.dumps({"what": "cuBLAS (torch.mm / torch.addmm, out_dtype = fp32) on the dW GEMM shapes, ~2 s back-to-back loops",
                      "config": {"workload": workload_name(args, cfg), "k": args.k, "slice_tokens": ts}, "rows": rows,
                      "peak_bf16_sustained_tflops": sus,
                      "frac_of_sustained_beta1": [r["beta1_tflops"] / sus for r in rows]}))
    return 0



def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--k", type=int, default=4)
    ap.add_argument("--axis", default="tokens", choices=["tokens", "ffn"],
                    help="split axis of the headline workload: token slices (north_star, default) or the paper-literal "
                         "ffn-axis split (osdp_ffn_split_mlp_*)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the per-k TFLOP/s and peak-bytes table")
    ap.add_argument("--graph", action="store_true",
                    help="also time the step captured in a CUDA graph and replayed (launch-bound configs: C1, C2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the table of BASELINE.json's other configurations (C1, C2, C3, C5 layer) in the default C4 line")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--granularity-sweep", default=None, metavar="H1,H2,...",
                    help="instead of the bench line: time and peak bytes vs split count for MLP operators of these "
                         "hidden sizes (ffn = 4 hidden, --sweep-tokens tokens), both split axes - the shape of the "
                         "paper's operator-splitting experiment (PAPER.md:231-247, Fig. 7)")
    ap.add_argument("--sweep-tokens", type=int, default=8192)
    ap.add_argument("--zdp", type=int, default=0, metavar="K",
                    help="instead of the bench line: ZDP mode with weight-slice gathering over the ranks torchrun started "
                         "(or one rank), K ffn slices (osdp_zdp_ffn_split_mlp_*, DESIGN.md section 11)")
    ap.add_argument("--stack", action="store_true",
                    help="with --config C5: instead of the bench line, run the 24-layer MLP stack with the split count "
                         "per layer chosen by osdp_plan from gamma/delta calibrated on this GPU (BASELINE.json config 5)")
    ap.add_argument("--slice-kernel-max-tiles", type=int, default=None, metavar="N",
                    help="set OSDP_TUNE_SLICE_KERNEL_MAX_TILES before the run (0 = one launch per GEMM for small slices too; "
                         "library default 128): the A/B of the one-kernel-per-slice path")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="osdp_set_tuning before the run, e.g. --tune mt2_min_k=2048 (keys: the OSDP_TUNE_* names of "
                         "include/osdp.h in lower case without the prefix); for A/B runs of the kernel-selection knobs")
    ap.add_argument("--vendor-dw", action="store_true",
                    help="instead of the bench line: the vendor library (cuBLAS through torch.mm / torch.addmm, fp32 output) "
                         "on the shapes of the dW GEMMs A5 / A6 of --config at --k, timed back to back for ~2 s each "
                         "(sustained, power-capped): the context for the dominant kernel's roofline fraction")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_2305_09940_b200 import inputs as I
    cfg = dict(I.CONFIGS[args.config])

    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        run_reference(args, cfg, rank)
        return 0

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the osdp-b200 hot path has no CPU fallback")
    from paper_2305_09940_b200 import binding as lib     # raises if the library was not built
    if args.slice_kernel_max_tiles is not None:
        lib.osdp_set_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, args.slice_kernel_max_tiles)
    for kv in args.tune:
        key, _, val = kv.partition("=")
        lib.osdp_set_tuning(getattr(lib, "OSDP_TUNE_" + key.strip().upper()), int(val))
    if args.granularity_sweep:
        return granularity_sweep(args, lib)
    if args.stack:
        return stack_bench(args, lib, cfg)
    if args.zdp:
        return zdp_bench(args, lib, cfg)
    if args.vendor_dw:
        return vendor_dw_bench(args, cfg)
    from paper_2305_09940_b200 import dist as D
    world, rank, local = D.init("nccl")
    peaks = load_peaks()
    T, h, f = cfg["tokens"], cfg["hidden"], cfg["ffn"]
    wl = Workload(lib, cfg, args.k, seed=D.rank_seed(cfg["seed"], rank))
    if args.axis != "tokens":
        wl.set_k(args.k, args.axis)
    flops = executed_flops(T, h, f)
    small = wl.resident_bytes() < 2 * L2_BYTES
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if small else None
    l2_note = "flush: 256 MiB memset between timed steps" if small else "inputs+outputs exceed L2 (126 MB); no flush"

    # ---- device-resident timing
    for _ in range(args.warmup):
        launches = wl.step()
    sampler = ClockSampler(local)
    sampler.start()
    ms_sum, wall_ms = timed_steps(wl.step, args.steps, world, flush)
    clocks = sampler.stop()
    ms_step = max_over_ranks(ms_sum / args.steps, world)
    ms_median = max_over_ranks(statistics.median(timed_steps.last), world)
    ms_min = max_over_ranks(min(timed_steps.last), world)
    value = world * flops / (ms_step * 1e-3) / 1e12
    graph = None
    if args.graph:
        g_ms, g_med, g_min = graph_step_ms(wl, args.steps, world, flush)
        g_ms = max_over_ranks(g_ms, world)
        graph = {"ms_per_step": g_ms, "ms_median": g_med, "ms_min": g_min, "value": world * flops / (g_ms * 1e-3) / 1e12,
                 "unit": UNIT, "how": "one step (forward + backward through the C ABI) captured in a CUDA graph, replayed"}

    # ---- per-launch trace of the same steps (CUDA events on the call's stream, inside the library)
    lib.osdp_trace_enable(True)
    for _ in range(args.steps):
        if flush is not None:
            flush.zero_()
        wl.step()
    trace = lib.osdp_trace_read()
    lib.osdp_trace_enable(False)
    per = {}
    for sid, ms in trace:
        per.setdefault(sid, []).append(ms)
    total_traced = sum(sum(v) for v in per.values())
    gemm_flops = 2.0 * T * h * f / args.k          # every GEMM launch of a slice: 2 T_s h f
    kernels = {}
    for sid, v in sorted(per.items()):
        avg = sum(v) / len(v)
        ent = {"step": lib.osdp_step_name(sid), "launches_per_step": len(v) // args.steps, "avg_ms": avg,
               "share": sum(v) / total_traced}
        if sid in GEMMS_PER_LAUNCH:
            ent["tflops"] = GEMMS_PER_LAUNCH[sid] * gemm_flops / (avg * 1e-3) / 1e12
        kernels[{21: "slice_fwd", 22: "slice_bwd", 10: "acc_to_out"}.get(sid, f"A{sid}")] = ent
    dom = max((s for s in per if s in GEMMS_PER_LAUNCH), key=lambda s: sum(per[s]))
    dom_avg = sum(per[dom]) / len(per[dom])
    gemm_flops *= GEMMS_PER_LAUNCH[dom]            # flops of one launch of the dominant kernel
    achieved = gemm_flops / (dom_avg * 1e-3) / 1e12
    peak = peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]) if cfg["dtype"] == "bf16" else None
    # DRAM bytes of the dominant kernel per launch, from the committed ncu --set full capture (profiles/traffic.json; its
    # .md names the command).  The dW GEMMs launch with beta = 0 on slice 0 (store only) and beta = 1 afterwards (fp32
    # read-modify-write): both are listed and `traffic` is the per-launch mean over the k launches of a step.
    traffic = traffic_detail = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath) and args.axis == "tokens":
        tj = json.load(open(tpath))
        key = f"{args.config}:k{args.k}:A{dom}"
        b0, b1 = tj.get(key + ":beta0"), tj.get(key + ":beta1")
        if b0 is not None and b1 is not None:
            traffic = (b0 + (args.k - 1) * b1) / args.k
            traffic_detail = {"beta0_launch": b0, "beta1_launch": b1, "launches_per_step": {"beta0": 1, "beta1": args.k - 1},
                              "source": tj.get("source")}
        elif tj.get(key) is not None:
            traffic = tj.get(key)
            traffic_detail = {"source": tj.get("source")}
    operand_path = None
    if os.path.exists(tpath) and args.axis == "tokens":
        l2b = json.load(open(tpath)).get(f"{args.config}:k{args.k}:A{dom}:l2_to_sm")
        if l2b and clocks.get("sm_mhz"):
            # what actually binds the 256 x 256-tile dW GEMMs: operand delivery L2 -> SM, whose
            # measured chip-wide ceiling is about 6300 B/clk (B300_MICROARCH.md "LTS throughput cap")
            bpc = l2b / (dom_avg * 1e-3 * clocks["sm_mhz"] * 1e6)
            operand_path = {"l2_to_sm_bytes_per_launch": l2b, "achieved_B_per_clk": bpc, "ceiling_B_per_clk": 6300.0,
                            "frac": bpc / 6300.0, "clock_mhz": clocks["sm_mhz"],
                            "how": "ncu lts__t_sectors_srcunit_tex_op_read x 32 B (profiles/r02_ncu_full.md) / (avg launch ms x SM clock sampled in this run)"}
    roofline = {"bound": "tensor", "kernel": f"{'mlp_slice_kernel' if dom >= 21 else 'gemm_bf16_sm100_kernel'} [{lib.osdp_step_name(dom)}]",
                "achieved": achieved, "peak": peak, "unit": UNIT, "frac": (achieved / peak) if peak else None,
                "traffic": traffic, "traffic_detail": traffic_detail, "operand_path": operand_path, "peak_source": f"{peaks['source']} (bf16_tflops_sustained: kernel timed inside a long step)",
                "frac_of_burst": achieved / peaks["bf16_tflops"], "frac_of_nominal": achieved / NOMINAL_BF16_TFLOPS,
                "flops_per_launch": gemm_flops, "avg_launch_ms": dom_avg,
                "how": "per-launch CUDA events recorded by the library on the call's stream over K traced steps"}
    if cfg["dtype"] != "bf16":
        ghz = (clocks.get("sm_mhz") or 1965.0) * 1e-3          # the clock sampled during the timed region
        alu_peak = 148 * 128 * 2 * ghz * 1e-3
        roofline.update({"bound": "alu", "kernel": f"gemm_f32_kernel [{lib.osdp_step_name(dom)}]", "peak": alu_peak,
                         "frac": achieved / alu_peak,
                         "peak_source": f"148 SMs x 128 FFMA/clk x 2 flop x {ghz:.3f} GHz (SM clock sampled in this run; fp32 FFMA path)"})

    # ---- end to end: host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        wl.step_e2e()
        torch.cuda.synchronize()
        e_sum, _ = timed_steps(wl.step_e2e, args.steps, world, None)
        serial_ms = max_over_ranks(e_sum / args.steps, world)
        e_ms = max_over_ranks(wl.run_e2e_pipelined(args.steps, world), world)
        e2e = {"value": world * flops / (e_ms * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": e_ms,
               "h2d_bytes_per_step": wl.h2d_bytes(), "d2h_bytes_per_step": wl.d2h_bytes(),
               "mode": "3 streams, double-buffered device tensors: H2D of step i+1 and D2H of step i-1 overlap the "
                       "kernels of step i; every step uploads all inputs and reads back all outputs",
               "serial_ms_per_step": serial_ms,
               "serial_value": world * flops / (serial_ms * 1e-3) / 1e12}

    # ---- per-k table: TFLOP/s and peak bytes vs the cost model (rank 0, N = 1 only)
    per_k = per_k_ffn = cost_fit = None
    if not args.no_sweep and world == 1 and cfg.get("ks"):
        tables = {"tokens": [], "ffn": []}       # "ffn": the paper-literal split (osdp_ffn_split_mlp_*), DESIGN.md section 10
        n_sw = max(3, args.steps // 2)
        for axis, tab in tables.items():
            for k in cfg["ks"]:
                wl.set_k(k, axis)
                for _ in range(2):
                    wl.step()
                s_ms, _ = timed_steps(wl.step, n_sw, 1, flush)
                s_ms /= n_sw
                tab.append({"k": k, "ms_per_step": s_ms, "tflops": flops / (s_ms * 1e-3) / 1e12,
                            "frac_of_sustained_peak": flops / (s_ms * 1e-3) / 1e12 / peak if peak else None})
        wl.set_k(args.k, args.axis)
        del wl
        torch.cuda.empty_cache()
        for axis, tab in tables.items():
            for ent in tab:
                ent["peak_bytes"] = measure_peak_bytes(lib, cfg, ent["k"], axis)
        per_k, per_k_ffn = tables["tokens"], tables["ffn"]
        cost_fit = {axis: fit_gamma_delta(tab) for axis, tab in tables.items()}
    configs = None
    if not args.no_configs and args.config == "C4" and world == 1:
        wl = None
        torch.cuda.empty_cache()
        configs = other_configs_table(lib, peaks, local)
    cpu = None
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        r = time_oracle(cfg, 1, 1)          # one untimed warm-up call, one timed
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "ms_per_step_median": ms_median, "ms_per_step_min": ms_min,
                "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
                "config": {"workload": workload_name(args, cfg), "tokens_per_gpu": T, "hidden": h, "ffn": f,
                           "k": args.k, "split_axis": args.axis, "flops_per_step": flops, "flops_counted": "14*T*h*f executed (12*T*h*f model)",
                           "l2": l2_note, "parallelism": f"dp{world} (independent token batches, no collective)",
                           "slice_kernel_max_tiles": lib.osdp_get_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES)},
                "value_model_flops_12x": value * 12.0 / 14.0,
                "frac_of_sustained_peak": value / world / peak if peak else None,
                "frac_of_nominal_peak": value / world / NOMINAL_BF16_TFLOPS,
                "frac_of_sustained_peak_note": "denominator = MEASURED_PEAKS.json bf16_tflops_sustained: the vendor (cuBLAS) bf16 GEMM "
                                               "timed inside a long run on this pool's B200s - a measured reference rate, not a hardware "
                                               "limit, so a fraction slightly above 1 (k = 1 rows) means the step ran faster than that GEMM",
                "clocks": clocks, "e2e": e2e, "graph": graph, "gpu_launches": int(launches) * args.steps,
                "roofline": roofline, "kernels": kernels, "per_k": per_k, "per_k_ffn_split": per_k_ffn, "cost_model_fit": cost_fit,
                "configs": configs, "cpu_baseline": cpu,
                "wall_ms_timed_region": wall_ms}
        print(json.dumps(line), flush=True)
    D.finalize()
    return 0


if __name__ == "__main__":
    sys.exit(main())
