#!/usr/bin/env python
"""bench.py -- fused SwiGLU-MLP TFLOP/s and % of roofline per M on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W [--workload qwen2.5-72b] [--impl reference]
    python bench.py --all            # every BASELINE.json point -> gpurun_out/results.{json,md}

A STEP is one pass of the whole hot path over one batch of synthetic input: for the
workload's (K, N) the fused entry point `swiglu_mlp` is called once per batch size M of that
BASELINE.json config.  The default workload is the largest single-GPU config, qwen2.5-72b
(BASELINE.json configs[4]: K = 8192, N = 29568, M = 8192, 4096, 1024, 128, 16, 1), which
exercises host dispatch, the small-M swap-AB/split-K kernel and the 1-CTA and 2-CTA tcgen05
kernels in every step.  `value` = sum(4*M*N*K) over the step / device time, inputs resident in
HBM (cold L2: 0.97 GB of weights per call).  `points` carries all 22 BASELINE.json points (five
shapes), each with its own timing, roofline fractions, on-device SM clock, unfused time and
mismatch counts against the oracle.  See DESIGN.md "Measurement".
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused_swiglu_mlp_tflops"
UNIT = "TFLOP/s"
NOMINAL = {"bf16_tflops": 2250.0, "hbm_gbs": 8000.0}
FALLBACK = {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0}
L2_BYTES = 126 << 20


def flops(M, N, K):
    return 4.0 * M * N * K                      # BASELINE.json: "TFLOP/s, counted as 4*M*N*K"


def algo_bytes(M, N, K):
    return 2 * K * N * 2 + M * K * 2 + M * N * 2  # BASELINE.json: weights + A + Y, once each


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return {"bf16_tflops": float(d["bf16_tflops"]),
                    "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    "hbm_gbs": float(d["hbm_gbs"])}, "measured"
        except Exception:
            pass
    return dict(FALLBACK), "fallback"


def roofline_time_s(M, N, K, peak_tflops, hbm_gbs):
    tc = flops(M, N, K) / (peak_tflops * 1e12)
    tm = algo_bytes(M, N, K) / (hbm_gbs * 1e9)
    return max(tc, tm), ("tensor" if tc >= tm else "hbm")


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region.

    NVML (nvidia_ml_py) polled every ~2 ms from a thread, so that even a timed region of a few
    milliseconds gets samples; falls back to `nvidia-smi -lms 50` if NVML is not importable."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []
        self.nvml, self.samples, self._stop = None, [], threading.Event()

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            idx = self.index
            if vis and all(v.strip().isdigit() for v in vis.split(",")):
                idx = int(vis.split(",")[self.index])
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.nvml = pynvml
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return self
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _poll(self):
        n = self.nvml
        while not self._stop.is_set():
            try:
                sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
                pw = n.nvmlDeviceGetPowerUsage(self.handle) / 1e3
                rs = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
                self.samples.append((sm, pw, rs))
            except Exception:
                pass
            time.sleep(0.002)

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    @staticmethod
    def _summary(sm, smax, power, reasons, how):
        # "under load": samples in the top half of the observed power range
        load = sm
        if power and max(power) > 1.5 * min(power):
            cut = (max(power) + min(power)) / 2
            load = [c for c, p in zip(sm, power) if p >= cut] or sm
        return {"sm_mhz": statistics.median(load) if load else None, "sm_max_mhz": smax,
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons),
                "samples": len(sm), "how": how}

    def stop(self):
        if self.nvml is not None:
            self._stop.set()
            self.thread.join(timeout=1)
            n = self.nvml
            bits = {"hw_slowdown": getattr(n, "nvmlClocksEventReasonHwSlowdown", 0x8),
                    "hw_thermal_slowdown": getattr(n, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                    "sw_thermal_slowdown": getattr(n, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                    "sw_power_cap": getattr(n, "nvmlClocksEventReasonSwPowerCap", 0x4)}
            reasons = {k for k, b in bits.items() for s in self.samples if s[2] & b}
            return self._summary([s[0] for s in self.samples], self.smax,
                                 [s[1] for s in self.samples], reasons, "nvml, 2 ms period")
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0, "how": "none"}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax = float(f[1]); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return self._summary(sm, smax, power, reasons, "nvidia-smi -lms 50")


# ---------------------------------------------------------------------------------------
# workload: one (K, N) shape with its batch sizes, resident in HBM, weights rotating
# ---------------------------------------------------------------------------------------
class Workload:
    def __init__(self, name, rank=0, rotate=True, Ms=None):
        import numpy as np
        import torch
        from paper_2607_02521_b200 import inputs
        table = dict(inputs.SHAPES)
        table.update(inputs.PAPER_SHAPES)
        self.name = name
        self.K, self.N, self.seed, self.Ms = table[name]
        if Ms:
            self.Ms = tuple(Ms)          # extra batch sizes for sweeps (same seeded streams)
        self.Mmax = max(self.Ms)
        K, N = self.K, self.N
        self.W1h, self.W2h = inputs.make_weights(K, N, self.seed)
        # rank r owns rows [r*Mmax, (r+1)*Mmax) of the shape's activation stream
        allA = inputs.make_activations((rank + 1) * self.Mmax, K, self.seed)
        self.Ah = np.ascontiguousarray(allA[rank * self.Mmax:])
        wbytes = 2 * K * N * 2
        self.copies = 1 if (not rotate or wbytes >= 2 * L2_BYTES) else -(-2 * L2_BYTES // wbytes) + 1
        to_dev = lambda b: torch.from_numpy(b.view(np.int16)).cuda().view(torch.bfloat16)
        self.W1 = [to_dev(self.W1h)]
        self.W2 = [to_dev(self.W2h)]
        self.A = [to_dev(self.Ah)]
        for _ in range(self.copies - 1):
            self.W1.append(self.W1[0].clone())
            self.W2.append(self.W2[0].clone())
            self.A.append(self.A[0].clone())
        self.Y = torch.empty((self.Mmax, N), dtype=torch.bfloat16, device="cuda")
        self.counter = 0
        self.l2_note = (f"cold L2: {self.copies} rotating copies of (A, W1, W2), "
                        f"{self.copies * wbytes / 2**20:.0f} MiB >= 2x L2" if self.copies > 1 else
                        f"weights {wbytes / 2**20:.0f} MiB per call exceed 2x L2")

    def call(self, fn, M, stream=None):
        """One C-ABI call with raw device pointers (fn = lib.swiglu_mlp or lib.swiglu_mlp_unfused)."""
        import torch
        c = self.counter % self.copies
        self.counter += 1
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        rc = fn(self.A[c].data_ptr(), self.W1[c].data_ptr(), self.W2[c].data_ptr(),
                self.Y.data_ptr(), M, self.N, self.K, stream)
        if rc != 0:
            from paper_2607_02521_b200 import binding
            raise binding.SwigluError(rc, binding.last_error())

    def unfused_fn(self, M):
        """swiglu_mlp_unfused_ex with a caller-owned Gate/Up workspace: the timing loop replays
        a captured CUDA graph, and the library's own per-stream workspace cannot be grown
        while a stream is capturing (include/swiglu_mlp.h)."""
        import torch
        from paper_2607_02521_b200 import binding as B
        lib = B.load()
        need = int(lib.swiglu_workspace_bytes(M, self.N, self.K, 1, -1))
        if getattr(self, "_ws", None) is None or self._ws.numel() < need:
            self._ws = torch.empty(max(need, 256), dtype=torch.uint8, device="cuda")
        ws = self._ws.data_ptr()

        def fn(a, w1, w2, y, m, n, k, stream):
            return lib.swiglu_mlp_unfused_ex(a, w1, w2, y, m, n, k, ws, need, -1, stream)
        return fn

    def fused_fn(self, variant=-1):
        """swiglu_mlp_ex with a caller-owned (zero-initialised) workspace: the timing loop replays
        a captured CUDA graph, and under capture the library does not create its own K-split
        workspace (include/swiglu_mlp.h) -- with the _ex form the captured calls run the same
        schedule (K-split last wave) an eager swiglu_mlp call does."""
        import torch
        from paper_2607_02521_b200 import binding as B
        lib = B.load()
        need = max(int(lib.swiglu_workspace_bytes(m, self.N, self.K, 0, v)) for v in (0, 1) for m in self.Ms)
        need = max(need, 256)
        if getattr(self, "_fws", None) is None or self._fws.numel() < need:
            self._fws = torch.zeros(need, dtype=torch.uint8, device="cuda")
        ws, nbytes = self._fws.data_ptr(), self._fws.numel()

        def fn(a, w1, w2, y, m, n, k, stream):
            return lib.swiglu_mlp_ex(a, w1, w2, y, m, n, k, ws, nbytes, variant, stream)
        return fn

    def flops_per_step(self):
        return sum(flops(M, self.N, self.K) for M in self.Ms)


def _capture(wl, fn, M, target_ms):
    """Warm `fn`, estimate its time, capture a whole number of weight-copy rotations of
    back-to-back calls into a CUDA graph.  Returns (graph, calls per replay, ms per replay)."""
    import torch
    for _ in range(3):
        wl.call(fn, M)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        wl.call(fn, M)
    e1.record()
    torch.cuda.synchronize()
    est_ms = max(e0.elapsed_time(e1) / 3, 1e-3)
    per = max(wl.copies, min(100, int(round(target_ms / est_ms))))
    per = -(-per // wl.copies) * wl.copies  # whole rotations: every replay starts at copy 0
    wl.counter = 0
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for _ in range(per):
            wl.call(fn, M)
    return g, per, est_ms * per


def _stats(samples, per, batches):
    med = statistics.median(samples)
    cv = (statistics.pstdev(samples) / med) if med > 0 else 0.0
    return {"us_median": med, "us_min": min(samples), "cv": cv, "calls_per_batch": per,
            "batches": batches}


_PROBE = None


def clock_probe():
    """Device buffer {SM cycles, ns} that CTA 0 of every GEMM-class launch of the library fills
    in (swiglu_set_clock_probe): cycles / ns = the SM clock that launch really ran at."""
    global _PROBE
    if _PROBE is None:
        import torch
        from paper_2607_02521_b200 import binding as B
        _PROBE = torch.zeros(2, dtype=torch.int64, device="cuda")
        B.swiglu_set_clock_probe(_PROBE)
    return _PROBE


def read_probe_mhz():
    c, ns = (int(v) for v in clock_probe().tolist())
    return (1e3 * c / ns) if ns > 0 else None


def time_points(wl, fns, M, target_ms=1.5, batches=15):
    """Median / min microseconds per call for each callable in `fns`, sampled INTERLEAVED
    (A, B, A, B, ...), so that clock / power / thermal drift during the measurement hits every
    candidate alike and ratios between them (speed-up over unfused) are not an artefact of
    order.  Each candidate is a batch of back-to-back calls (rotating weight copies) captured
    once into a CUDA graph and replayed between two CUDA events: what a serving loop replaying
    a captured decode step sees, free of Python launch gaps.  `sm_mhz` is the SM clock of the
    last GEMM-class launch of each replay, measured on the device (clock64 / globaltimer)."""
    import torch
    probe = clock_probe()
    caps = [_capture(wl, fn, M, target_ms) for fn in fns]
    for g, per, ms in caps:
        for _ in range(max(2, int(10.0 / max(ms, 1e-3)))):   # ~10 ms of warm replays each
            g.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    samples = [[] for _ in fns]
    mhz = [[] for _ in fns]
    for _ in range(batches):
        for i, (g, per, _) in enumerate(caps):
            probe.zero_()
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            samples[i].append(e0.elapsed_time(e1) * 1e3 / per)
            f = read_probe_mhz()
            if f:
                mhz[i].append(f)
    out = []
    for i, smp in enumerate(samples):
        st = _stats(smp, caps[i][1], batches)
        st["sm_mhz"] = round(statistics.median(mhz[i]), 0) if mhz[i] else None
        st["sm_mhz_min"] = round(min(mhz[i]), 0) if mhz[i] else None
        out.append(st)
    return out


def time_point(wl, fn, M, target_ms=1.5, batches=15):
    """One callable (see time_points)."""
    return time_points(wl, [fn], M, target_ms, batches)[0]


def check_point(wl, M, max_rows=128):
    """Mismatch counts of both paths against the CPU oracle on sampled rows (tests/ holds the
    parity tests proper; this is the count the north_star asks to report beside the timing).
    Rows: both ends of every 32-lane TMEM quarter of every 128-row tile (inputs.sample_rows),
    thinned evenly to `max_rows` only where that is more (M >= 4096: still >= 2 rows of each of
    the 64 row tiles at M = 8192); all N columns of each row."""
    import numpy as np
    import torch
    import oracle
    from paper_2607_02521_b200 import binding as B, check, inputs
    rows = inputs.sample_rows(M)
    if len(rows) > max_rows:
        idx = np.linspace(0, len(rows) - 1, max_rows).round().astype(int)
        rows = rows[idx]
    y_ref, _ = oracle.swiglu_oracle_rows(wl.Ah[:M], wl.W1h, wl.W2h, rows)
    out = {}
    sel = torch.from_numpy(rows).cuda()
    lib = B.load()
    for key, fn in (("fused", lib.swiglu_mlp), ("unfused", lib.swiglu_mlp_unfused)):
        wl.Y[:M].fill_(float("nan"))
        wl.call(fn, M)
        c = (wl.counter - 1) % wl.copies
        assert c < wl.copies  # all copies hold the same bits as wl.Ah / wl.W1h / wl.W2h
        torch.cuda.synchronize()
        y = wl.Y[:M][sel].view(torch.int16).cpu().numpy().view(np.uint16)
        rep = check.compare(y, y_ref)
        out[key] = {"mismatches": rep.mismatches, "checked": rep.checked,
                    "max_ratio": round(rep.max_ratio, 4), "not_rne_of_ref": rep.not_rne_of_ref}
    return out


ABLATION_MIN_M = 256   # BW_eff / fusion efficiency are defined on M >= 256 profiles


def measure_points(wl, peaks, do_check=True, Ms=None, isolated=False):
    import torch
    from paper_2607_02521_b200 import binding as B
    lib = B.load()
    pts = []
    for M in (Ms or wl.Ms):
        f, u = time_points(wl, [wl.fused_fn(), wl.unfused_fn(M)], M)
        t = f["us_median"] * 1e-6
        fl, by = flops(M, wl.N, wl.K), algo_bytes(M, wl.N, wl.K)
        t_roof, bound = roofline_time_s(M, wl.N, wl.K, peaks["bf16_tflops"], peaks["hbm_gbs"])
        t_nom, _ = roofline_time_s(M, wl.N, wl.K, NOMINAL["bf16_tflops"], NOMINAL["hbm_gbs"])
        t_sus, _ = roofline_time_s(M, wl.N, wl.K, peaks["bf16_tflops_sustained"], peaks["hbm_gbs"])
        uv = B.swiglu_selected_variant(M, wl.N, wl.K, unfused=True)
        p = {"workload": wl.name, "M": M, "N": wl.N, "K": wl.K,
             "variant": B.swiglu_variant_name(B.swiglu_selected_variant(M, wl.N, wl.K)),
             "us": round(f["us_median"], 2), "us_min": round(f["us_min"], 2), "cv": round(f["cv"], 4),
             "sm_mhz": f["sm_mhz"], "sm_mhz_min": f["sm_mhz_min"],
             "tflops": round(fl / t / 1e12, 2), "gbs": round(by / t / 1e9, 1), "bound": bound,
             "roofline_frac": round(t_roof / t, 4), "roofline_frac_nominal": round(t_nom / t, 4),
             "roofline_frac_sustained": round(t_sus / t, 4),
             "unfused_variant": B.swiglu_variant_name(uv, unfused=True),
             "unfused_us": round(u["us_median"], 2), "unfused_cv": round(u["cv"], 4),
             "speedup_vs_unfused": round(u["us_median"] / f["us_median"], 3)}
        if isolated:
            # one call at a time, device idle before it (no PDL overlap with a predecessor)
            p["us_isolated"] = round(time_isolated(wl, lib.swiglu_mlp, M), 2)
        if M >= ABLATION_MIN_M:
            # Fusion-efficiency ablation (Table 6): the standalone
            # elementwise stage gives BW_eff; eta = saved time / (4*M*N*2 bytes / BW_eff).
            gu = torch.empty((2, M, wl.N), dtype=torch.bfloat16, device="cuda").normal_()

            def ew(a, w1, w2, y, m, n, k, stream, _g=gu[0].data_ptr(), _u=gu[1].data_ptr()):
                return lib.swiglu_silu_mul(_g, _u, y, m * n, stream)
            e = time_point(wl, ew, M)
            bw_eff = 6.0 * M * wl.N / (e["us_median"] * 1e-6)        # bytes/s: read G, U, write Y
            saved = (u["us_median"] - f["us_median"]) * 1e-6
            p["elementwise_us"] = round(e["us_median"], 2)
            p["swiglu_share_of_unfused"] = round(e["us_median"] / u["us_median"], 4)
            p["bw_eff_gbs"] = round(bw_eff / 1e9, 1)
            p["fusion_efficiency"] = round(saved / (8.0 * M * wl.N / bw_eff), 3)
            del gu
        if do_check:
            p["parity"] = check_point(wl, M)
        pts.append(p)
    return pts


def time_isolated(wl, fn, M, reps=30):
    """Median microseconds of ONE eager call with the device idle before it (sync on both
    sides, CUDA events): no programmatic-dependent-launch overlap with a predecessor."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    out = []
    for _ in range(reps + 3):
        torch.cuda.synchronize()
        e0.record()
        wl.call(fn, M)
        e1.record()
        torch.cuda.synchronize()
        out.append(e0.elapsed_time(e1) * 1e3)
    return statistics.median(out[3:])


# ---------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------
_W_CACHE = {}


def oracle_sample(name, rows, nthreads=0):
    """Time the oracle, as it stands, on the first `rows` rows of the workload's largest batch
    (all N columns, all of K).  Returns (seconds, flops, threads)."""
    import oracle
    from paper_2607_02521_b200 import inputs
    table = dict(inputs.SHAPES)
    table.update(inputs.PAPER_SHAPES)
    K, N, seed, Ms = table[name]
    if name not in _W_CACHE:
        _W_CACHE[name] = inputs.make_weights(K, N, seed)
        oracle.swiglu_oracle(inputs.make_activations(1, K, seed), *_W_CACHE[name], nthreads)
    W1, W2 = _W_CACHE[name]
    A = inputs.make_activations(rows, K, seed)
    t0 = time.perf_counter()
    _, used = oracle.swiglu_oracle(A, W1, W2, nthreads)
    dt = time.perf_counter() - t0
    return dt, flops(rows, N, K), used


def cpu_baseline(name, target_s=12.0):
    dt, fl, used = oracle_sample(name, 16)
    rows = int(max(16, min(2048, 16 * target_s / max(dt, 1e-3))))
    dt, fl, used = oracle_sample(name, rows)
    table_rows = rows
    return {"value": round(fl / dt / 1e12, 6), "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"{table_rows} rows x all N columns of {name} (fp64 oracle, "
                      f"{fl / 1e9:.1f} GFLOP counted as 4MNK) in {dt:.2f} s",
            "seconds": round(dt, 3)}


def run_reference(args, ranks):
    """--impl reference: this tier's reference arm is the CPU oracle, timed as it stands."""
    if ranks.rank != 0:
        return
    name = args.workload
    dt, fl, used = oracle_sample(name, 16)
    budget_s = float(os.environ.get("SWIGLU_REFERENCE_BUDGET_S", "60"))   # whole run, CPU seconds
    rows = int(max(8, min(1024, 16 * (budget_s / max(1, args.steps + args.warmup)) / max(dt, 1e-3))))
    times = []
    for i in range(args.warmup + args.steps):
        dt, fl, used = oracle_sample(name, rows)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * sum(times) / len(times)
    value = fl / (ms * 1e-3) / 1e12
    sample = f"{rows} rows x all N columns of {name} per step (fp64 CPU oracle)"
    from paper_2607_02521_b200 import inputs
    table = dict(inputs.SHAPES)
    table.update(inputs.PAPER_SHAPES)
    K, N, _, Ms = table[name]
    workload = f"{name}: K={K}, N={N}, one swiglu_mlp call per M in {sorted(Ms, reverse=True)}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(value, 6), "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms, 3), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload, "sample": sample},
        "cpu_baseline": {"value": round(value, 6), "unit": UNIT, "cores": used,
                         "kind": "oracle", "sample": sample},
        "e2e": {"value": round(value, 6), "unit": UNIT, "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------
def read_traffic(name, M, kernel=None):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, copied
    from the committed `ncu --set full` captures (profiles/traffic.csv names the summary each
    row comes from), or (None, None) when that (workload, M) has not been captured."""
    import csv
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        hit = None
        for row in csv.DictReader(open(path)):
            if row["workload"] == name and int(row["M"]) == int(M) and (
                    kernel is None or row["kernel"] == kernel):
                hit = row                                   # the last (newest) row wins
        if hit:
            return int(hit["dram_bytes_read"]) + int(hit["dram_bytes_write"]), hit["source"]
    except Exception:
        pass
    return None, None


def run_ours(args, ranks):
    import numpy as np
    import torch
    from paper_2607_02521_b200 import binding as B, inputs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(ranks.local_rank)
    lib = B.load()
    peaks, peak_src = load_peaks()
    wl = Workload(args.workload, rank=ranks.rank)
    order = sorted(wl.Ms, reverse=True)          # largest batch first: the host runs ahead
    Mdom = order[0]
    launches_per_step = sum(B.swiglu_launches_per_call(M, wl.N, wl.K) for M in order)
    probe = clock_probe()

    def step(ev=None):
        for M in order:
            if ev is not None and M == Mdom:
                ev[0].record()
                wl.call(lib.swiglu_mlp, M)
                ev[1].record()
            else:
                wl.call(lib.swiglu_mlp, M)

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    dom_events = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                  for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(ranks.local_rank).start()
    ranks.barrier()
    torch.cuda.synchronize()
    e0.record()
    for i in range(args.steps):
        step(dom_events[i])
    e1.record()
    torch.cuda.synchronize()
    ranks.barrier()
    clocks = sampler.stop()
    ms_total = ranks.max_over_ranks(e0.elapsed_time(e1))
    ms_per_step = ms_total / args.steps
    value = wl.flops_per_step() * ranks.world / (ms_per_step * 1e-3) / 1e12
    dom_ms = statistics.mean(a.elapsed_time(b) for a, b in dom_events)
    # SM clock inside the dominant kernel, measured on the device (one more launch of it)
    probe.zero_()
    wl.call(lib.swiglu_mlp, Mdom)
    torch.cuda.synchronize()
    clocks["sm_mhz_in_dominant_kernel"] = round(read_probe_mhz() or 0.0, 0) or None
    clocks["in_kernel_how"] = "clock64 / %globaltimer of CTA 0 (swiglu_set_clock_probe)"

    # roofline of the dominant kernel (the largest-M call: a dense bf16 contraction)
    t_roof, bound = roofline_time_s(Mdom, wl.N, wl.K, peaks["bf16_tflops"], peaks["hbm_gbs"])
    long_run = ms_total >= 1000.0      # a kernel timed inside a long step: sustained figure
    if bound == "tensor":
        achieved, runit = flops(Mdom, wl.N, wl.K) / (dom_ms * 1e-3) / 1e12, "TFLOP/s"
        peak = peaks["bf16_tflops_sustained"] if long_run else peaks["bf16_tflops"]
    else:
        achieved, peak, runit = algo_bytes(Mdom, wl.N, wl.K) / (dom_ms * 1e-3) / 1e9, peaks["hbm_gbs"], "GB/s"
    traffic, traffic_src = read_traffic(
        wl.name, Mdom, B.swiglu_variant_name(B.swiglu_selected_variant(Mdom, wl.N, wl.K)))
    roofline = {"bound": bound, "achieved": round(achieved, 2), "peak": peak, "unit": runit,
                "frac": round(achieved / peak, 4), "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes": algo_bytes(Mdom, wl.N, wl.K),
                "algorithmic_flops": flops(Mdom, wl.N, wl.K),
                "kernel": B.swiglu_variant_name(B.swiglu_selected_variant(Mdom, wl.N, wl.K)),
                "M": Mdom, "us_per_launch": round(dom_ms * 1e3, 2),
                "share_of_step": round(dom_ms / ms_per_step, 4),
                "peak_source": (f"{peak_src} MEASURED_PEAKS.json, "
                                f"{'sustained' if long_run and bound == 'tensor' else 'burst'} figure "
                                f"(timed region {ms_total:.0f} ms)") if peak_src == "measured"
                               else "fallback (B200_PROFILING.md)",
                "frac_of_burst": round(achieved / peaks["bf16_tflops"], 4) if bound == "tensor" else None,
                "frac_of_sustained": round(achieved / peaks["bf16_tflops_sustained"], 4) if bound == "tensor" else None,
                "frac_of_nominal": round(achieved / (NOMINAL["bf16_tflops"] if bound == "tensor" else NOMINAL["hbm_gbs"]), 4)}

    # end to end through the C ABI with HOST buffers (pinned): every step uploads that step's
    # inputs (the weights once, every batch of activations) and downloads every Y.
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).pin_memory()
        hW1, hW2 = pin(wl.W1h), pin(wl.W2h)
        hAs = [pin(wl.Ah[:M]) for M in order]
        hYs = [torch.empty((M, wl.N), dtype=torch.int16).pin_memory() for M in order]
        stream = torch.cuda.current_stream().cuda_stream

        def e2e_step():
            B.swiglu_mlp_host_batched(hAs, hYs, order, hW1, hW2, wl.N, wl.K, stream=stream)

        h2d = sum(M * wl.K * 2 for M in order) + 2 * wl.K * wl.N * 2
        d2h = sum(M * wl.N * 2 for M in order)
        # bound the leg to ~10 s of PCIe traffic (a 72B step moves 2 GB)
        e2e_steps = max(3, min(args.steps, 20, int(10.0 * 40e9 / (h2d + d2h))))
        e2e_step()
        ranks.barrier()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(e2e_steps):
            e2e_step()
        e1.record()
        torch.cuda.synchronize()
        ranks.barrier()
        e2e_ms = ranks.max_over_ranks(e0.elapsed_time(e1)) / e2e_steps
        e2e = {"value": round(wl.flops_per_step() * ranks.world / (e2e_ms * 1e-3) / 1e12, 3), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": round(e2e_ms, 3),
               "steps": e2e_steps,
               "api": "swiglu_mlp_host_batched (pinned host buffers; weights uploaded once per step in "
                      "column chunks, uploads / kernels / downloads pipelined)",
               "pcie_gbs": round((h2d + d2h) / (e2e_ms * 1e-3) / 1e9, 1)}
        # sampled check of what came back over PCIe: rows spread over every batch and, in the
        # largest batch, over the whole range of row tiles
        if ranks.rank == 0 and not args.no_check:
            import oracle
            from paper_2607_02521_b200 import check
            bad = checked = 0
            for bi, M in enumerate(order):
                rows = inputs.sample_rows(M)
                cap = 16 if bi == 0 else 2
                if len(rows) > cap:
                    rows = rows[np.linspace(0, len(rows) - 1, cap).round().astype(int)]
                y_ref, _ = oracle.swiglu_oracle_rows(wl.Ah[:M], wl.W1h, wl.W2h, rows)
                rep = check.compare(hYs[bi].numpy().view(np.uint16)[rows], y_ref)
                bad += rep.mismatches
                checked += rep.checked
            e2e["mismatches"], e2e["checked"] = bad, checked
        del hW1, hW2, hAs, hYs

    points, cpu = None, None
    if ranks.rank == 0:
        if ranks.world == 1 and not args.no_cpu_baseline:
            cpu = cpu_baseline(wl.name)
        if not args.no_points:
            # all 22 BASELINE.json points: the headline shape first (its inputs are resident),
            # then the other four shapes, each with its own cold-L2 rotation
            names = [wl.name] + [n for n in inputs.SHAPES if n != wl.name]
            if args.points == "headline":
                names = [wl.name]
            points = []
            for name in names:
                w = wl if name == wl.name else Workload(name, rank=0)
                points += measure_points(w, peaks, do_check=not args.no_check, isolated=True)
                if w is not wl:
                    del w
                    torch.cuda.empty_cache()
            order_key = {n: i for i, n in enumerate(inputs.SHAPES)}
            points.sort(key=lambda q: (order_key.get(q["workload"], 99), q["M"]))
    ranks.barrier()
    if ranks.rank != 0:
        return
    out = {
        "metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": ranks.world,
        "steps": args.steps, "warmup": warmup, "ms_per_step": round(ms_per_step, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": f"{wl.name}: K={wl.K}, N={wl.N}, one swiglu_mlp call per M in {order}",
                   "l2": wl.l2_note, "parallelism": f"replicas x{ranks.world} (no collective)",
                   "flops_per_step": wl.flops_per_step(),
                   "points": "all 22 BASELINE.json (shape, M) points, each timed on its own"
                             if points is not None and args.points == "all" else args.points},
        "clocks": clocks, "roofline": roofline,
        "gpu_launches": launches_per_step * args.steps,
    }
    if e2e is not None:
        out["e2e"] = e2e
    if cpu is not None:
        out["cpu_baseline"] = cpu
    if points is not None:
        out["points"] = points
        out["points_summary"] = {
            "count": len(points),
            "mismatches_fused": sum(q["parity"]["fused"]["mismatches"] for q in points if "parity" in q),
            "mismatches_unfused": sum(q["parity"]["unfused"]["mismatches"] for q in points if "parity" in q),
            "min_roofline_frac": min(q["roofline_frac"] for q in points),
            "points_at_or_above_0.70_of_measured_roofline": sum(q["roofline_frac"] >= 0.70 for q in points),
            "min_speedup_vs_unfused": min(q["speedup_vs_unfused"] for q in points)}
    print(json.dumps(out))


def points_table(pts):
    hdr = ("| workload | M | variant | us | SM MHz | TFLOP/s | GB/s | bound | % of measured roofline | "
           "% of nominal | us isolated | unfused us | speed-up | elementwise us (share of unfused) | "
           "fusion eff. | mismatches fused / unfused (checked) |")
    lines = [hdr, "|" + "---|" * 16]
    for p in pts:
        par = p.get("parity")
        ptxt = (f"{par['fused']['mismatches']} / {par['unfused']['mismatches']} ({par['fused']['checked']})"
                if par else "-")
        ew = (f"{p['elementwise_us']} ({100 * p['swiglu_share_of_unfused']:.0f} %)"
              if "elementwise_us" in p else "-")
        lines.append(f"| {p['workload']} | {p['M']} | {p['variant']} | {p['us']} | {p.get('sm_mhz') or '-'} | "
                     f"{p['tflops']} | {p['gbs']} | {p['bound']} | {100 * p['roofline_frac']:.1f} | "
                     f"{100 * p['roofline_frac_nominal']:.1f} | {p.get('us_isolated', '-')} | "
                     f"{p['unfused_us']} | {p['speedup_vs_unfused']} | {ew} | "
                     f"{p.get('fusion_efficiency', '-')} | {ptxt} |")
    return "\n".join(lines)


def run_all(args):
    """Every BASELINE.json point (and, with --paper-grid, the paper's own grid) -> a table."""
    import torch
    from paper_2607_02521_b200 import inputs
    peaks, peak_src = load_peaks()
    names = list(inputs.SHAPES) + (list(inputs.PAPER_SHAPES) if args.paper_grid else [])
    if args.only:
        names = [n for n in names if n in args.only.split(",")]
    sampler = ClockSampler(0).start()
    pts = []
    for name in names:
        wl = Workload(name)
        pts += measure_points(wl, peaks, do_check=not args.no_check, isolated=True)
        del wl
        torch.cuda.empty_cache()
    clocks = sampler.stop()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    json.dump({"peaks": peaks, "peak_source": peak_src, "clocks": clocks, "points": pts},
              open(os.path.join(ROOT, "gpurun_out", "results.json"), "w"), indent=1)
    md = points_table(pts)
    open(os.path.join(ROOT, "gpurun_out", "results.md"), "w").write(md + "\n")
    print(md)
    print(json.dumps({"clocks": clocks, "peak_source": peak_src}))


def run_decode_study(args):
    """Decode-size anatomy (`--decode-study`): per (shape, M <= 128), microseconds per call in a
    CUDA-graph chain (cold L2, rotating weight copies) of
      * the launch-floor probe (the decode kernel's launch with an empty body),
      * swiglu_mlp (plain [K,N] weights),
      * swiglu_mlp_packed (prepacked W_fused: one TMA box per stage, weight loads ahead of
        griddepcontrol.wait),
      * swiglu_mlp_unfused,
    plus the isolated (device idle before the call) time of the two fused forms.
    Writes gpurun_out/decode_study.md."""
    import torch
    from paper_2607_02521_b200 import binding as B, inputs
    lib = B.load()
    peaks, _ = load_peaks()
    table = list(inputs.SHAPES) + list(inputs.PAPER_SHAPES)
    names = [n for n in table if n in args.only.split(",")] if args.only else list(inputs.SHAPES)
    Ms = [int(m) for m in args.sweep_m.split(",") if int(m) <= 128]
    lines = ["| workload | M | HBM roofline us | floor probe us | fused us | packed us | unfused us | "
             "fused isolated us | packed isolated us | fused % of roofline | packed % of roofline |",
             "|" + "---|" * 11]
    for name in names:
        wl = Workload(name, Ms=Ms)
        nbytes = B.swiglu_packed_weight_bytes(wl.N, wl.K)
        Wp = [torch.empty(nbytes // 2, dtype=torch.int16, device="cuda") for _ in range(wl.copies)]
        for c in range(wl.copies):
            B.swiglu_pack_weights(wl.W1[c], wl.W2[c], Wp[c], wl.N, wl.K)
        torch.cuda.synchronize()
        ptrs = {wl.W1[c].data_ptr(): Wp[c].data_ptr() for c in range(wl.copies)}

        def packed(a, w1, w2, y, m, n, k, stream):
            return lib.swiglu_mlp_packed(a, ptrs[w1], y, m, n, k, stream)

        for M in Ms:
            probe_fn = lib.swiglu_launch_floor_probe
            res = time_points(wl, [probe_fn, lib.swiglu_mlp, packed, wl.unfused_fn(M)], M,
                              batches=args.sweep_batches)
            iso_f = time_isolated(wl, lib.swiglu_mlp, M)
            iso_p = time_isolated(wl, packed, M)
            t_roof, _ = roofline_time_s(M, wl.N, wl.K, peaks["bf16_tflops"], peaks["hbm_gbs"])
            us = [r["us_median"] for r in res]
            lines.append(f"| {name} | {M} | {t_roof * 1e6:.2f} | {us[0]:.2f} | {us[1]:.2f} | {us[2]:.2f} | "
                         f"{us[3]:.2f} | {iso_f:.2f} | {iso_p:.2f} | {100 * t_roof * 1e6 / us[1]:.1f} | "
                         f"{100 * t_roof * 1e6 / us[2]:.1f} |")
            print(lines[-1], flush=True)
        del wl, Wp
        torch.cuda.empty_cache()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    open(os.path.join(ROOT, "gpurun_out", "decode_study.md"), "w").write("\n".join(lines) + "\n")


def run_fp8(args):
    """FP8-operand table (`--fp8`): per BASELINE.json (shape, M) the FP8
    (E4M3) fused call next to the bf16 fused call on the same shape -- microseconds (cold L2,
    CUDA-graph replay, interleaved sampling), TFLOP/s (4MNK), fraction of the FP8 roofline
    max(4MNK / (2 x measured bf16 peak), (2KN + MK + 2MN bytes) / HBM) -- the guide's nominal
    fp8 : bf16 = 2 ratio applied to the measured bf16 peak -- and mismatches against the fp64 FP8
    oracle on sampled rows.  Writes gpurun_out/fp8_results.md."""
    import numpy as np
    import torch
    import oracle
    from paper_2607_02521_b200 import binding as B, check, inputs
    lib = B.load()
    peaks, peak_src = load_peaks()
    names = [n for n in inputs.SHAPES if not args.only or n in args.only.split(",")]
    lines = ["| workload | M | variant | fp8 us | fp8 TFLOP/s | fp8 GB/s | bound | % of fp8 roofline "
             "(2 x measured bf16 peak) | SM MHz | bf16 fused us | fp8 speed-up over bf16 | "
             "mismatches (checked) |", "|" + "---|" * 12]
    for name in names:
        wl = Workload(name)
        K, N = wl.K, wl.N
        A8h, W1h, W2h, sg, su = inputs.make_fp8_case(wl.Mmax, N, K, seed=50 + wl.seed)
        wbytes = 2 * K * N
        copies = 1 if wbytes >= 2 * L2_BYTES else -(-2 * L2_BYTES // wbytes) + 1
        up = lambda x: torch.from_numpy(x).cuda()
        A8 = [up(A8h) for _ in range(copies)]
        W1 = [up(W1h) for _ in range(copies)]
        W2 = [up(W2h) for _ in range(copies)]
        ctr = [0]

        def fp8(a, w1, w2, y, m, n, k, stream):
            c = ctr[0] % copies
            ctr[0] += 1
            return lib.swiglu_mlp_fp8(A8[c].data_ptr(), W1[c].data_ptr(), W2[c].data_ptr(), y, m, n, k,
                                      sg, su, stream)
        for M in wl.Ms:
            f8, f16 = time_points(wl, [fp8, wl.fused_fn()], M, batches=args.sweep_batches)
            t = f8["us_median"] * 1e-6
            fl = flops(M, N, K)
            by = 2 * K * N + M * K + M * N * 2
            tc, tm = fl / (2 * peaks["bf16_tflops"] * 1e12), by / (peaks["hbm_gbs"] * 1e9)
            rows = inputs.sample_rows(M)
            if len(rows) > 32:
                rows = rows[np.linspace(0, len(rows) - 1, 32).round().astype(int)]
            y_ref, _ = oracle.swiglu_oracle_fp8(A8h[:M], W1h, W2h, sg, su, rows=rows)
            wl.Y[:M].fill_(float("nan"))
            rc = lib.swiglu_mlp_fp8(A8[0].data_ptr(), W1[0].data_ptr(), W2[0].data_ptr(), wl.Y.data_ptr(),
                                    M, N, K, sg, su, torch.cuda.current_stream().cuda_stream)
            assert rc == 0, B.last_error()
            torch.cuda.synchronize()
            y = wl.Y[:M][torch.from_numpy(rows).cuda()].view(torch.int16).cpu().numpy().view(np.uint16)
            rep = check.compare(y, y_ref)
            lines.append(f"| {name} | {M} | {B.swiglu_variant_name(B.swiglu_selected_variant(M, N, K))} | "
                         f"{f8['us_median']:.2f} | {fl / t / 1e12:.1f} | {by / t / 1e9:.0f} | "
                         f"{'tensor' if tc >= tm else 'hbm'} | {100 * max(tc, tm) / t:.1f} | {f8['sm_mhz'] or '-'} | "
                         f"{f16['us_median']:.2f} | {f16['us_median'] / f8['us_median']:.3f} | "
                         f"{rep.mismatches} ({rep.checked}) |")
            print(lines[-1], flush=True)
        del wl, A8, W1, W2
        torch.cuda.empty_cache()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    open(os.path.join(ROOT, "gpurun_out", "fp8_results.md"), "w").write("\n".join(lines) + "\n")
    print(json.dumps({"peak_source": peak_src, "fp8_peak_tflops": 2 * peaks["bf16_tflops"]}))


def run_ncu_points(args):
    """`--ncu-points name:M[:u][,name:M...]`: the kernels behind the per-point claims, launched
    eagerly so that `ncu -k regex:... --set full` can capture them one by one: per point one
    warm-up call and one more of swiglu_mlp (":u" adds swiglu_mlp_unfused, ":p" the prepacked
    form, ":8" the FP8 form, ":v" -- as labelled CONTEXT only -- the vendor GEMM torch.matmul(A,
    [W1|W2]) on the same operands).  Weight copies rotate as in the timed runs (cold L2).  Prints one
    line per point with the CUDA-event time of the last call -- NOT a bench value when run
    under a profiler."""
    import torch
    from paper_2607_02521_b200 import binding as B, inputs
    lib = B.load()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    cache = {}
    specs = [sp.split(":") for sp in args.ncu_points.split(",")]
    for parts in specs:
        name, M, flags = parts[0], int(parts[1]), "".join(parts[2:])
        if name not in cache:
            cache.clear()
            torch.cuda.empty_cache()
            cache[name] = Workload(name, Ms=[int(q[1]) for q in specs if q[0] == name])
        wl = cache[name]
        fns = [("fused", lib.swiglu_mlp)]
        if "u" in flags:
            fns.append(("unfused", lib.swiglu_mlp_unfused))
        if "p" in flags:
            nbytes = B.swiglu_packed_weight_bytes(wl.N, wl.K)
            Wp = torch.empty(nbytes // 2, dtype=torch.int16, device="cuda")
            B.swiglu_pack_weights(wl.W1[0], wl.W2[0], Wp, wl.N, wl.K)
            fns.append(("packed", lambda a, w1, w2, y, m, n, k, st, _w=Wp: lib.swiglu_mlp_packed(
                a, _w.data_ptr(), y, m, n, k, st)))
        if "8" in flags:
            A8h, W1h, W2h, sg, su = inputs.make_fp8_case(M, wl.N, wl.K, seed=50 + wl.seed)
            A8, W18, W28 = (torch.from_numpy(x).cuda() for x in (A8h, W1h, W2h))
            fns.append(("fp8", lambda a, w1, w2, y, m, n, k, st, _t=(A8, W18, W28, sg, su): lib.swiglu_mlp_fp8(
                _t[0].data_ptr(), _t[1].data_ptr(), _t[2].data_ptr(), y, m, n, k, _t[3], _t[4], st)))
        if "v" in flags:
            Wcat = torch.cat([wl.W1[0], wl.W2[0]], dim=1).contiguous()
            GU = torch.empty((M, 2 * wl.N), dtype=torch.bfloat16, device="cuda")

            def vendor(a, w1, w2, y, m, n, k, st, _w=Wcat, _o=GU, _a=wl.A[0]):
                torch.matmul(_a[:m], _w, out=_o)
                return 0
            fns.append(("context: vendor GEMM", vendor))
        for label, fn in fns:
            for i in range(2):
                torch.cuda.synchronize()
                e0.record()
                wl.call(fn, M)
                e1.record()
                torch.cuda.synchronize()
            print(f"{name} M={M} {label}: {e0.elapsed_time(e1) * 1e3:.1f} us (eager, second of 2 calls)", flush=True)


def run_sustained(args):
    """`--sustained name:M[,name:M...]`: throughput under SUSTAINED load (each candidate runs back
    to back for ~1.5 s, so the 1 kW power cap, not the burst clock, sets the SM clock; then the
    next ~40 ms are timed), candidates interleaved over three rounds:
      * swiglu_mlp (fused), swiglu_mlp_unfused,
      * CONTEXT ONLY: the vendor GEMM (torch.matmul -> cuBLAS) on the same A and the
        concatenated [K, 2N] weights -- the same 4MNK FLOP, WITHOUT the activation, writing
        twice the output.  It is what MEASURED_PEAKS.json's bf16 figures are made of, measured
        here on the same box, shape, data and protocol.  Not part of the product path.
    Also repeated with all-zero operands (same kernels, minimal switching power): when the two
    agree there, what separates them on random data is energy per FLOP, not schedule.
    Writes gpurun_out/sustained.md."""
    import torch
    from paper_2607_02521_b200 import binding as B, inputs
    import pynvml
    pynvml.nvmlInit()
    h = pynvml.nvmlDeviceGetHandleByIndex(0)
    lib = B.load()
    probe = clock_probe()
    st = torch.cuda.current_stream().cuda_stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    lines = ["| workload | M | operands | candidate | us (3 rounds) | TFLOP/s (median) | SM MHz in kernel | power W |",
             "|" + "---|" * 8]
    for spec in args.sustained.split(","):
        name, M = spec.split(":")[0], int(spec.split(":")[1])
        table = dict(inputs.SHAPES)
        table.update(inputs.PAPER_SHAPES)
        K, N, seed, _ = table[name]
        fl = flops(M, N, K)
        for data in ("N(0,1) x N(0,0.02)", "zeros"):
            g = torch.Generator(device="cuda").manual_seed(seed)
            if data == "zeros":
                A = torch.zeros((M, K), device="cuda", dtype=torch.bfloat16)
                Wcat = torch.zeros((K, 2 * N), device="cuda", dtype=torch.bfloat16)
            else:
                A = torch.randn((M, K), device="cuda", generator=g).bfloat16()
                Wcat = (torch.randn((K, 2 * N), device="cuda", generator=g) * 0.02).bfloat16()
            W1, W2 = Wcat[:, :N].contiguous(), Wcat[:, N:].contiguous()
            Y = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
            GU = torch.empty((M, 2 * N), dtype=torch.bfloat16, device="cuda")
            ptr = (A.data_ptr(), W1.data_ptr(), W2.data_ptr(), Y.data_ptr(), M, N, K, st)
            cands = {"swiglu_mlp (fused)": lambda: lib.swiglu_mlp(*ptr),
                     "swiglu_mlp_unfused": lambda: lib.swiglu_mlp_unfused(*ptr),
                     "context: cuBLAS GEMM A.[W1|W2] (no activation)": lambda: torch.matmul(A, Wcat, out=GU)}
            auto = B.swiglu_selected_variant(M, N, K)
            for v in range(B.swiglu_num_variants()):   # the other large-M kernels, forced
                vn = B.swiglu_variant_name(v)
                if M > 256 and v != auto and vn.startswith("fused_2cta"):
                    cands[f"forced variant {vn}"] = (lambda _v=v: lib.swiglu_mlp_ex(*ptr[:7], None, 0, _v, st))
            res = {k: [] for k in cands}
            for fn in cands.values():
                for _ in range(3):
                    fn()
            torch.cuda.synchronize()
            reps = max(4, int(40e-3 / (fl / 1.3e15)))
            for rnd in range(3):
                for nm, fn in cands.items():
                    t_end = time.time() + 1.5
                    pw = []
                    while time.time() < t_end:
                        for _ in range(4):
                            fn()
                        torch.cuda.synchronize()
                        pw.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1e3)
                    probe.zero_()
                    e0.record()
                    for _ in range(reps):
                        fn()
                    e1.record()
                    torch.cuda.synchronize()
                    res[nm].append((e0.elapsed_time(e1) * 1e3 / reps,
                                    None if nm.startswith("context") else read_probe_mhz(),
                                    statistics.median(pw)))
            for nm, v in res.items():
                us = [x[0] for x in v]
                mhz = [x[1] for x in v if x[1]]
                lines.append(f"| {name} | {M} | {data} | {nm} | {', '.join(f'{u:.0f}' for u in us)} | "
                             f"{fl / statistics.median(us) / 1e6:.0f} | "
                             f"{(f'{statistics.median(mhz):.0f}' if mhz else '-')} | "
                             f"{statistics.median([x[2] for x in v]):.0f} |")
                print(lines[-1], flush=True)
            del A, Wcat, W1, W2, Y, GU
            torch.cuda.empty_cache()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    open(os.path.join(ROOT, "gpurun_out", "sustained.md"), "w").write("\n".join(lines) + "\n")


def run_sweep(args):
    """Dispatch-table sweeps (`--sweep variants` / `--sweep ksplit`): time every fused variant
    (forced through swiglu_mlp_ex) or every split-K factor of the small-M kernel
    (SWIGLU_KSPLIT) per (shape, M), cold L2, CUDA-graph replay.  Writes a markdown table to
    gpurun_out/sweep_<kind>.md; select_fused() / smallm_ksplit() in swiglu_api.cu are fitted
    to these tables."""
    import torch
    from paper_2607_02521_b200 import binding as B, inputs
    lib = B.load()
    table = list(inputs.SHAPES) + list(inputs.PAPER_SHAPES)
    names = [n for n in table if n in args.only.split(",")] if args.only else list(inputs.SHAPES)
    Ms = [int(m) for m in args.sweep_m.split(",")]
    nvar = B.swiglu_num_variants()
    lines = []
    if args.sweep == "variants":
        cols = ["auto"] + [B.swiglu_variant_name(v) for v in range(nvar)]
        lines += ["| workload | M | " + " | ".join(cols) + " | auto picks |", "|---|---|" + "---|" * (len(cols) + 1)]
    else:
        ks = list(range(1, 9))
        lines += ["| workload | M | " + " | ".join(f"S={k}" for k in ks) + " | auto (S) |", "|---|---|" + "---|" * 9]

    def forced(v):
        return lambda *a: forced.wl.fused_fn(v)(*a)

    def usable(fn, wl, M):
        try:
            wl.call(fn, M)
            return True
        except B.SwigluError:
            return False

    for name in names:
        wl = Workload(name, Ms=Ms)
        forced.wl = wl
        for M in Ms:
            if args.sweep == "variants":
                # every variant of this (shape, M) sampled INTERLEAVED, so clock / power drift
                # hits all of them alike
                cand = [v for v in [-1] + list(range(nvar)) if usable(forced(v), wl, M)]
                res = dict(zip(cand, time_points(wl, [forced(v) for v in cand], M, batches=args.sweep_batches)))
                cells = [f"{res[v]['us_median']:.2f}" if v in res else "n/a" for v in [-1] + list(range(nvar))]
                pick = B.swiglu_variant_name(B.swiglu_selected_variant(M, wl.N, wl.K))
            else:
                # SWIGLU_KSPLIT is baked in when a call is captured, so capture one graph per S
                small = [v for v in range(nvar) if "smallm" in B.swiglu_variant_name(v)][0]
                cells = []
                for k in ks + [0]:
                    os.environ["SWIGLU_KSPLIT"] = str(k)
                    B.swiglu_reload_env()
                    try:
                        cells.append(f"{time_point(wl, forced(small), M)['us_median']:.2f}")
                    except B.SwigluError:
                        cells.append("n/a")
                os.environ.pop("SWIGLU_KSPLIT", None)
                B.swiglu_reload_env()
                pick = cells.pop()
            lines.append(f"| {name} | {M} | " + " | ".join(cells) + f" | {pick} |")
            print(lines[-1], flush=True)
        del wl
        torch.cuda.empty_cache()
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    open(os.path.join(ROOT, "gpurun_out", f"sweep_{args.sweep}.md"), "w").write("\n".join(lines) + "\n")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="qwen2.5-72b")
    ap.add_argument("--points", default="all", choices=["all", "headline"],
                    help="which shapes the per-point table covers (all = the 22 BASELINE.json points)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--all", action="store_true")
    ap.add_argument("--paper-grid", action="store_true")
    ap.add_argument("--only", default="")
    ap.add_argument("--no-points", action="store_true")
    ap.add_argument("--no-check", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", default="", choices=["", "variants", "ksplit"])
    ap.add_argument("--sweep-m", default="1,16,32,64,128,256")
    ap.add_argument("--sweep-batches", type=int, default=15)
    ap.add_argument("--decode-study", action="store_true")
    ap.add_argument("--fp8", action="store_true")
    ap.add_argument("--ncu-points", default="")
    ap.add_argument("--sustained", default="")
    args = ap.parse_args()
    from paper_2607_02521_b200.dist import Ranks
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        if rank != 0:
            return                      # rank 0 alone runs the CPU oracle
        class _Solo:
            rank, world, local_rank = 0, 1, 0
        run_reference(args, _Solo())
        return
    if args.all:
        run_all(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.decode_study:
        run_decode_study(args)
        return
    if args.fp8:
        run_fp8(args)
        return
    if args.ncu_points:
        run_ncu_points(args)
        return
    if args.sustained:
        run_sustained(args)
        return
    ranks = Ranks()
    if ranks.world != args.gpus and ranks.rank == 0:
        print(f"note: --gpus {args.gpus} but WORLD_SIZE={ranks.world}; launch with torchrun",
              file=sys.stderr)
    try:
        run_ours(args, ranks)
    finally:
        ranks.close()


if __name__ == "__main__":
    main()
