#!/usr/bin/env python
"""bench.py -- throughput of the batched 4x4 Birkhoff projection (forward + backward) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config2|config3_s10|config3_s30|
                    config3_s100|config4|config5] [--impl ours|reference] [--no-cpu-baseline]
    N > 1:  python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
                --master-port P bench.py --gpus N --steps K --warmup W

A STEP is one pass of the whole hot path (F0-F8 forward kernel, then B0-B4 backward kernel) over
one batch of B synthetic matrices.  Default workload = BASELINE.json configs[1]: B = 2^20 fp32 matrices, H and
dL/dP iid N(0,1), tol 1e-6, max_iter 20.  Rank r of N works on its own B matrices (weak scaling, no data-path
collective: SURVEY.md 8(e)); the only cross-rank traffic is the max over ranks of the measured time.

L2: every rank rotates over `sets` distinct buffer sets (H, P, dP, dH; >= 1 GiB in total, L2 is 126 MB); step i
runs forward on set i % sets and backward on set (i+1) % sets, whose P was written sets-1 steps earlier, so
backward reads P from HBM as it does in training, where the rest of the network runs in between.

ONE compact JSON line on stdout (rank 0; contract_line(), under 2 KB: the driver keeps a bounded tail of stdout).
The full result (every other BASELINE.json config under `workloads`, the SURVEY.md 8(f) widenings, histograms)
goes to gpurun_out/bench_detail.json and, as one line, to stderr; `per_config` in the stdout line carries
[step us, forward frac, backward frac, max Err] of each other config.
`value` = matrices/s through forward+backward with inputs resident in HBM: the median over --regions regions of K
steps each between two CUDA events on the launching stream (max over ranks); `value_single` = the one K-step region
bracketed by barrier + synchronize; `roofline.isolated_us` = the forward launched alone after an L2-displacing
write (no overlap with a neighbouring launch), `roofline.avg_us` = back to back; `e2e` = the same through the
host-buffer C-ABI call birkhoff4_forward_backward_host (pinned host memory in, P and dH back out, copies inside
the timed region); `roofline_kernels` = each kernel's average launch duration (K back-to-back launches of that
kernel over the same rotation between two events) against the measured HBM copy bandwidth (MEASURED_PEAKS.json),
`roofline` = the slower of the two, `traffic` = ncu DRAM bytes per launch from profiles/traffic.csv;
`fwd.update_histogram` = share of matrices by number of Newton updates (BASELINE.json configs[2] asks for it);
`cpu_baseline` = the fp64 oracle timed on this host on a bounded sample (a reported baseline, not the target).
`--impl reference` times that oracle alone (rank 0 only); the oracle is test infrastructure and is imported
nowhere else in this file's GPU path.
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "4x4 projections/sec fwd+bwd"
UNIT = "matrices/s"
FWD_BYTES, BWD_BYTES = 128, 192            # algorithmic HBM bytes per matrix; bf16 logits: 96 forward
WORKLOADS = {
    "config2": dict(config=2, B=1 << 20, scale=1.0, max_iter=20, desc="B=2^20 fp32, H,dP iid N(0,1)"),
    "config3_s10": dict(config=3, B=1 << 20, scale=10.0, max_iter=32, desc="B=2^20 fp32, H iid N(0,10^2)"),
    "config3_s30": dict(config=3, B=1 << 20, scale=30.0, max_iter=32, desc="B=2^20 fp32, H iid N(0,30^2)"),
    "config3_s100": dict(config=3, B=1 << 20, scale=100.0, max_iter=32, desc="B=2^20 fp32, H iid N(0,100^2)"),
    "config4": dict(config=4, B=1 << 24, scale=2.0, max_iter=20, desc="B=2^24, H bf16(N(0,4)), P,dP,dH fp32"),
    "config5": dict(config=5, B=1 << 22, scale=None, max_iter=32, desc="B=2^22 fp32 heterogeneous (BASELINE configs[4])"),
}
TOL = 1e-6


# ------------------------------------------------------------------------------------------------ inputs
def make_inputs(wl, rank, k):
    """seeded synthetic H (fp32, or bf16 bit patterns) and G for buffer set k of rank `rank`"""
    from paper_2606_07574_b200 import inputs
    sub = 100 * rank + k
    c, B = wl["config"], wl["B"]
    if c == 2:
        return inputs.normal(B, 1.0, config=2, sub=sub)
    if c == 3:
        return inputs.normal(B, wl["scale"], config=3, sub=1000 * int(wl["scale"]) + sub)
    if c == 4:
        H, G = inputs.normal(B, 2.0, config=4, sub=sub)
        return inputs.f32_to_bf16_bits(H), G
    H, G, _ = inputs.heterogeneous(B, config=5, sub=sub)
    return H, G


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock and throttle reasons sampled with NVML while the timed regions run"""
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTED = {"sw_power_cap": 0x4}

    def __init__(self, index):
        self.samples, self.reasons, self.h, self.nv = [], set(), None, None
        self._stop, self._on, self._thread = threading.Event(), threading.Event(), None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:                                                               # CUDA_VISIBLE_DEVICES may renumber
                self.h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(index).uuid))
            except Exception:                                                  # noqa: BLE001
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self._reasons = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        except Exception:                                                      # noqa: BLE001 (no NVML: report nulls)
            self.max_mhz, self.h = None, None

    def sample(self):
        if self.h is None:
            return
        try:
            self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
            r = self._reasons(self.h)
            for name, bit in {**self.BAD, **self.NOTED}.items():
                if r & bit:
                    self.reasons.add(name)
        except Exception:                                                      # noqa: BLE001
            pass

    def _run(self):
        while not self._stop.is_set():
            if self._on.is_set():
                self.sample()
            time.sleep(0.004)

    def start(self):
        self._thread = threading.Thread(target=self._run, daemon=True)
        self._thread.start()

    def region(self, on):
        (self._on.set if on else self._on.clear)()

    def stop(self):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ peaks
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _finite(x):
    """strict JSON: NaN/Inf (e.g. the Sinkhorn-20 baseline's error at s >= 30, where exp underflows) become null"""
    if isinstance(x, float):
        return x if np.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _finite(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_finite(v) for v in x]
    return x


# ------------------------------------------------------------------------------------------------ the contract line
LINE_LIMIT = 2048       # bytes: the driver keeps a bounded tail of stdout, so the one JSON line must stay small


def _r(x, nd=4):
    """numbers rounded to `nd` significant digits (the detail file keeps full precision)"""
    if isinstance(x, float):
        return float("%.*g" % (nd, x)) if np.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _r(v, nd) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_r(v, nd) for v in x]
    return x


def contract_line(full):
    """the ONE stdout line: the contract keys of the full result only, under LINE_LIMIT bytes.  Everything else
    (per-workload blocks, widenings, histograms) goes to the detail file and to stderr."""
    rf = full["roofline"]
    line = {k: full[k] for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                                 "scaling", "vs_baseline", "dtype", "data")}
    line["value_single"] = full.get("value_single")
    c = full["config"]
    line["config"] = {k: c[k] for k in ("workload", "desc", "B_per_gpu", "tol", "max_iter", "l2") if k in c}
    line["roofline"] = {k: rf.get(k) for k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "avg_us", "isolated_us",
                                               "frac_isolated", "bytes_per_launch", "traffic", "peak_source")}
    wr = rf.get("work_roofline") or {}
    line["roofline"]["work_bound"], line["roofline"]["work_frac"] = wr.get("bound"), wr.get("frac")   # slower of HBM / FP32 / SFU work
    line["roofline_step"] = {k: full["roofline_step"].get(k) for k in ("bound", "achieved", "peak", "unit", "frac")}
    line["fwd_us"], line["bwd_us"] = full["fwd"]["us"]["median"], full["bwd"]["us"]["median"]
    line["bwd_frac"] = full["roofline_kernels"]["backward_kernel"]["frac"]
    line["max_marginal_err"] = full["max_marginal_err"]
    line["mean_newton_updates"] = full["fwd"]["mean_newton_updates"]
    if full.get("cpu_baseline"):
        line["cpu_baseline"] = {k: full["cpu_baseline"][k] for k in ("value", "unit", "cores", "kind", "sample")}
    e = full["e2e"]
    line["e2e"] = {k: e[k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "steps", "api")}
    line["clocks"] = full.get("clocks")
    line["gpu_launches"] = full.get("gpu_launches")
    if full.get("workloads"):
        # name: [step_us, forward frac of HBM peak, backward frac, max marginal error, forward frac of the work roofline]
        line["per_config"] = {n: [w["step_us"]["median"], w["roofline_kernels"]["forward_kernel"]["frac"],
                                  w["roofline_kernels"]["backward_kernel"]["frac"], w["max_marginal_err"],
                                  (w["roofline_kernels"]["forward_kernel"].get("work_roofline") or {}).get("frac")]
                              for n, w in full["workloads"].items() if "@" not in n}
    if full.get("detail_file"):
        line["detail_file"] = full["detail_file"]
    line = _r(_finite(line))
    text = json.dumps(line, separators=(",", ":"))
    if len(text) > LINE_LIMIT:                                                 # never the case today; keep the contract keys
        for k in ("per_config", "detail_file", "roofline_step", "value_single"):
            line.pop(k, None)
        text = json.dumps(line, separators=(",", ":"))
    return text


def write_detail(full):
    """the full result: gpurun_out/bench_detail.json when that folder can be written, and one line on stderr"""
    text = json.dumps(_finite(full))
    path = None
    try:
        d = os.path.join(ROOT, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        path = os.path.join(d, "bench_detail.json")
        with open(path, "w") as f:
            f.write(text + "\n")
        path = os.path.relpath(path, ROOT)
    except OSError:
        path = None
    print(text, file=sys.stderr)
    return path


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_step(oracle, H, G, nthreads=0):
    P = oracle.forward(H, nthreads=nthreads)
    return oracle.backward(P, G, nthreads=nthreads)


def run_reference(args, wl):
    """the fp64 CPU oracle as it stands, on a bounded sample of the workload per step (rank 0 only)"""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_2606_07574_b200 import inputs
    # bounded sample per step: about 2^20 (N(0,1)-like) or 2^16 (slow-Sinkhorn regimes) matrices over the whole run
    budget = (1 << 16) if wl["config"] in (3, 5) else (1 << 20)
    n = max(64, min(wl["B"], 1 << 14, budget // max(1, args.steps + args.warmup)))
    H, G = make_inputs(dict(wl, B=n), 0, 0)
    if wl["config"] == 4:
        H = inputs.bf16_bits_to_f32(H)
    for _ in range(args.warmup):
        oracle_step(oracle, H, G)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(oracle, H, G)
    dt = time.perf_counter() - t0
    v = n * args.steps / dt
    sample = "first %d matrices of the workload per step, forward (Sinkhorn-Knopp to 1e-14 + certified fallback) + backward (KKT solve), fp64" % n
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "desc": wl["desc"], "B_per_step": n, "tol": 1e-14},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------ our arm
def _rooflines(B, bf16, f_us, b_us, s_us, peak, peak_src, workload, mean_updates, sm_mhz, n_sm):
    """per-kernel and per-step achieved HBM bandwidth against the measured copy peak, and the forward's second
    roofline (instruction issue, from the ncu instruction count of this workload under profiles/)"""
    fb = 96 if bf16 else FWD_BYTES
    nominal = 7700.0                                                           # B200_PROFILING.md: HGX nominal HBM3e GB/s
    k = {}
    for name, us, byts in (("forward_kernel", f_us, fb), ("backward_kernel", b_us, BWD_BYTES)):
        ach = B * byts / (us["median"] * 1e-6) / 1e9
        k[name] = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                   "frac_min_time": B * byts / (us["min"] * 1e-6) / 1e9 / peak, "frac_of_nominal_7700": ach / nominal,
                   "avg_us": us["median"], "min_us": us["min"], "bytes_per_launch": B * byts,
                   "traffic": ncu_traffic(name, workload)}
        if k[name]["frac"] > 1.0:
            k[name]["note"] = "above 1: the measured copy peak underestimates what a pure stream reaches"
    ach = B * (fb + BWD_BYTES) / (s_us["median"] * 1e-6) / 1e9
    step = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "bytes_per_step": B * (fb + BWD_BYTES),
            "peak_source": peak_src}
    # north_star's roofline: the slower of the bytes at HBM peak and the executed exp / FMA work at SFU / FP32 peak
    # (128 FP32 lanes and 16 SFU lanes per clock per SM: B200_PROFILING.md), counts per 32 matrices from the ncu SASS
    # opcode tables (profiles/traffic.csv).  Unlike issue_diagnostic below it does not count selects, min/max, votes,
    # shared-memory moves: what separates the kernel from this floor is exactly that overhead plus imperfect overlap.
    work = ncu_work("forward_kernel", workload)
    if work:
        clk = n_sm * sm_mhz * 1e6
        t = {"hbm": B * fb / (peak * 1e9) * 1e6, "fp32": work[0] * B / (128.0 * clk) * 1e6, "sfu": work[1] * B / (16.0 * clk) * 1e6}
        bound = max(t, key=t.get)
        k["forward_kernel"]["work_roofline"] = {
            "bound": bound, "floor_us": t[bound], "frac": t[bound] / f_us["median"], "hbm_us": t["hbm"], "fp32_us": t["fp32"],
            "sfu_us": t["sfu"], "fp32_warp_instr_per_32": work[0], "mufu_warp_instr_per_32": work[1],
            "peak_source": "nominal: 128 FP32 and 16 SFU lanes per clock per SM x %d SMs x %d MHz; HBM: %s" % (n_sm, sm_mhz, peak_src)}
    winst = ncu_warp_inst("forward_kernel", workload)
    if winst:
        issue_peak = 4.0 * n_sm * sm_mhz * 1e6                                 # warp instructions / s
        ach_i = winst * (B / 32.0) / (f_us["median"] * 1e-6)
        k["forward_kernel"]["issue_diagnostic"] = {
            "bound": "alu", "achieved": ach_i / 1e12, "peak": issue_peak / 1e12, "unit": "T warp-instr/s", "frac": ach_i / issue_peak,
            "warp_instr_per_32_matrices": winst, "source": "ncu smsp__inst_executed.sum of this workload (profiles/traffic.csv)",
            "peak_source": "nominal: 4 issue slots per clock per SM x %d SMs x %d MHz (half-rate instructions hold a slot for "
                           "two clocks, profiles/r2_pipe_microbench.md: the attainable fraction is below 1)" % (n_sm, sm_mhz)}
    return k, step


def ncu_work(kernel, workload):
    """(FP32, MUFU) warp instructions per 32 matrices of `kernel` on `workload` from profiles/traffic.csv, or None"""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            k = [x.strip() for x in line.split(",")]
            if len(k) >= 7 and k[0] == kernel and k[1] == workload:
                return float(k[5]), float(k[6])
    return None


def ncu_warp_inst(kernel, workload):
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            k = [x.strip() for x in line.split(",")]
            if len(k) >= 5 and k[0] == kernel and k[1] == workload:
                return float(k[4])
    return None


def ncu_traffic(kernel, workload):
    """dram bytes per launch of `kernel` on `workload` from the committed ncu --set full summaries, or None"""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            k = [x.strip() for x in line.split(",")]
            if len(k) >= 4 and k[0] == kernel and k[1] == workload:
                return float(k[2]) + float(k[3])
    return None


class Timer:
    """R timed regions of K calls each, CUDA events on the launching (current) stream; per-call us: median and min"""

    def __init__(self, torch, K, R):
        self.torch, self.K, self.R = torch, K, R

    def __call__(self, fn):
        t = self.torch
        per = []
        for _ in range(self.R):
            e0, e1 = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(self.K):
                fn(i)
            e1.record()
            e1.synchronize()
            per.append(e0.elapsed_time(e1) * 1e3 / self.K)
        return {"median": statistics.median(per), "min": min(per), "regions": self.R, "calls_per_region": self.K}


def isolated_us(torch, fn, n=20):
    """one launch alone between two events, after a 256 MiB write has displaced L2 (126 MB): median us over n.
    No back-to-back overlap (programmatic dependent launch) helps this figure; it includes the launch's own ramp and tail."""
    flush = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
    per = []
    for i in range(n):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn(i)
        e1.record()
        e1.synchronize()
        per.append(e0.elapsed_time(e1) * 1e3)
    del flush
    return statistics.median(per)


def err_stats(torch, P):
    """Err of PAPER.md:323 in fp64 on the stored fp32 P: max, mean, and the largest single marginal deviation"""
    mx, sm, einf, n = 0.0, 0.0, 0.0, P.shape[0]
    for lo in range(0, n, 1 << 22):
        P64 = P[lo:lo + (1 << 22)].double()
        r, c = (P64.sum(2) - 1).abs(), (P64.sum(1) - 1).abs()
        e = r.sum(1) + c.sum(1)
        mx, sm = max(mx, float(e.max())), sm + float(e.sum())
        einf = max(einf, float(r.max()), float(c.max()))
        del P64, r, c, e
    return {"max_marginal_err": mx, "mean_marginal_err": sm / n, "max_err_inf": einf}


def measure_workload(torch, bk, inputs, name, wl, rank, K, R, peak, peak_src, sm_mhz, n_sm, max_iter=None, sort_by_class=False):
    """device-resident measurement of one workload: forward, backward and step timings, accuracy, histogram"""
    B, bf16 = wl["B"], wl["config"] == 4
    max_iter = wl["max_iter"] if max_iter is None else max_iter
    set_bytes = B * (32 if bf16 else 64) + 3 * B * 64
    nsets = max(2, -(-(1 << 30) // set_bytes))                                 # >= 1 GiB in rotation (L2 is 126 MB)
    distinct = 1 if B > (1 << 21) else nsets                                   # large B: one draw, copied (host time)
    sets = []
    for k in range(nsets):
        if k < distinct:
            if wl["config"] == 5:
                H, G, _ = inputs.heterogeneous(B, config=5, sub=100 * rank + k, sort_by_class=sort_by_class)
            else:
                H, G = make_inputs(wl, rank, k)
            H0, G0 = (H, G) if k == 0 else (H0, G0)
        Hd = torch.from_numpy(H.view(np.int16)).cuda().view(torch.bfloat16) if bf16 else torch.from_numpy(H).cuda()
        sets.append(dict(H=Hd, G=torch.from_numpy(G).cuda(), P=torch.empty((B, 4, 4), device="cuda"),
                         dH=torch.empty((B, 4, 4), device="cuda")))
    fwd = bk.birkhoff4_forward_bf16 if bf16 else bk.birkhoff4_forward

    def f_call(i):
        s = sets[i % nsets]
        fwd(s["H"], s["P"], TOL, max_iter)

    def b_call(i):
        t = sets[i % nsets]
        bk.birkhoff4_backward(t["P"], t["G"], t["dH"])

    def step(i):
        s, t = sets[i % nsets], sets[(i + 1) % nsets]
        fwd(s["H"], s["P"], TOL, max_iter)
        bk.birkhoff4_backward(t["P"], t["G"], t["dH"])

    for i in range(nsets):                                                     # every set has a valid P before backward reads it
        f_call(i)
    for i in range(3):
        step(i)
    torch.cuda.synchronize()
    timer = Timer(torch, K, R)
    s_us, f_us, b_us = timer(step), timer(f_call), timer(b_call)
    f_iso = isolated_us(torch, f_call)
    acc = err_stats(torch, sets[0]["P"])
    hist = torch.zeros(64, dtype=torch.int64, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    (bk.birkhoff4_forward_bf16_ex if bf16 else bk.birkhoff4_forward_ex)(sets[0]["H"], sets[0]["P"], TOL, max_iter,
                                                                        hist=hist, n_unconverged=unc)
    h = hist.cpu().numpy()
    mean_updates = float((h * np.arange(64)).sum() / max(h.sum(), 1))
    kern, step_roof = _rooflines(B, bf16, f_us, b_us, s_us, peak, peak_src, name, mean_updates, sm_mhz, n_sm)
    kern["forward_kernel"]["isolated_us"] = f_iso
    kern["forward_kernel"]["frac_isolated"] = B * (96 if bf16 else FWD_BYTES) / (f_iso * 1e-6) / 1e9 / peak
    res = {"desc": wl["desc"] + (", sorted by class" if sort_by_class else ""), "B": B, "max_iter": max_iter,
           "value": B / (s_us["median"] * 1e-6), "unit": UNIT, "step_us": s_us, "forward_us": f_us, "backward_us": b_us,
           "fwd_matrices_per_s": B / (f_us["median"] * 1e-6), "roofline_step": step_roof, "roofline_kernels": kern,
           "mean_newton_updates": mean_updates,
           "update_histogram": {str(k): round(float(h[k]) / max(h.sum(), 1), 6) for k in range(64) if h[k]},
           "unconverged": int(unc.item()), "buffer_sets": nsets, **acc}
    return res, sets, (H0, G0)


def measure_widenings(torch, bk, inputs, K, R, peak):
    """fused forward+backward, n = 8, general OT, fused mix: per-call us and achieved HBM GB/s"""
    timer = Timer(torch, K, R)
    out = {}
    B = 1 << 20
    H, G = inputs.normal(B, 1.0, config=2)
    sets = [dict(H=torch.from_numpy(H).cuda() + 0 * k, G=torch.from_numpy(G).cuda(), P=torch.empty((B, 4, 4), device="cuda"),
                 dH=torch.empty((B, 4, 4), device="cuda")) for k in range(4)]
    for want_P, byts in ((True, 256), (False, 192)):
        us = timer(lambda i: bk.birkhoff4_forward_backward(sets[i % 4]["H"], sets[i % 4]["G"], sets[i % 4]["P"] if want_P else None,
                                                           sets[i % 4]["dH"], TOL, 20, want_P=want_P))
        out["fused_forward_backward" + ("" if want_P else "_no_P")] = {
            "desc": "B=2^20 N(0,1), one kernel, P %s" % ("written" if want_P else "not written"), "us": us,
            "bytes_per_matrix": byts, "achieved_GBs": B * byts / (us["median"] * 1e-6) / 1e9,
            "frac": B * byts / (us["median"] * 1e-6) / 1e9 / peak, "matrices_per_s": B / (us["median"] * 1e-6)}
    del sets
    B8 = 1 << 18
    for s in (1.0, 10.0):
        H8, G8 = inputs.normal_n(B8, 8, s, config=8)
        s8 = [dict(H=torch.from_numpy(H8).cuda() + 0 * k, G=torch.from_numpy(G8).cuda(), P=torch.empty((B8, 8, 8), device="cuda"),
                   dH=torch.empty((B8, 8, 8), device="cuda")) for k in range(4)]
        fus = timer(lambda i: bk.birkhoff8_forward(s8[i % 4]["H"], s8[i % 4]["P"], 2e-6, 60))
        bus = timer(lambda i: bk.birkhoff8_backward(s8[i % 4]["P"], s8[i % 4]["G"], s8[i % 4]["dH"]))
        P64 = s8[0]["P"].double()
        err = float(((P64.sum(2) - 1).abs().sum(1) + (P64.sum(1) - 1).abs().sum(1)).max())
        out["birkhoff8_s%g" % s] = {
            "desc": "B=2^18 fp32 8x8, H iid N(0,%g^2)" % s, "forward_us": fus, "backward_us": bus, "max_marginal_err": err,
            "forward": {"bytes_per_matrix": 512, "frac": B8 * 512 / (fus["median"] * 1e-6) / 1e9 / peak,
                        "matrices_per_s": B8 / (fus["median"] * 1e-6)},
            "backward": {"bytes_per_matrix": 768, "frac": B8 * 768 / (bus["median"] * 1e-6) / 1e9 / peak,
                         "matrices_per_s": B8 / (bus["median"] * 1e-6)}}
        del s8, P64
    Bo = 1 << 20
    Cm, a, b, Go = inputs.ot_problem(Bo, 4, 4, 2.0, config=9)
    so = [dict(C=torch.from_numpy(Cm).cuda() + 0 * k, a=torch.from_numpy(a).cuda(), b=torch.from_numpy(b).cuda(),
               G=torch.from_numpy(Go).cuda(), T=torch.empty((Bo, 4, 4), device="cuda"), D=torch.empty((Bo, 4, 4), device="cuda"))
          for k in range(4)]
    fus = timer(lambda i: bk.entropic_ot_forward(so[i % 4]["C"], so[i % 4]["a"], so[i % 4]["b"], so[i % 4]["T"], 0.7, 2e-6, 60))
    bus = timer(lambda i: bk.entropic_ot_backward(so[i % 4]["T"], so[i % 4]["G"], so[i % 4]["D"], 0.7))
    out["entropic_ot_4x4"] = {"desc": "B=2^20 4x4 costs N(0,2^2), Gamma(4) marginals, eta = 0.7", "forward_us": fus, "backward_us": bus,
                              "forward": {"bytes_per_matrix": 160, "frac": Bo * 160 / (fus["median"] * 1e-6) / 1e9 / peak},
                              "backward": {"bytes_per_matrix": 192, "frac": Bo * 192 / (bus["median"] * 1e-6) / 1e9 / peak}}
    del so
    Bm, C = 1 << 16, 1024
    Hm = torch.from_numpy(inputs.normal(Bm, 1.0, config=2, sub=7)[0]).cuda()
    g = torch.Generator(device="cuda").manual_seed(inputs.SEED + 77)
    Xs = [torch.randn((Bm, 4, C), device="cuda", generator=g).bfloat16() for _ in range(2)]
    Ys = [torch.empty_like(x) for x in Xs]
    us = timer(lambda i: bk.birkhoff4_forward_mix(Hm, Xs[i % 2], Ys[i % 2], None, TOL, 20))
    byts = 64 + 2 * 4 * C * 2
    out["fused_mix_bf16"] = {"desc": "B=2^16 tokens, 4 streams x C=1024 bf16: Y = proj(exp(H)) X in one kernel", "us": us,
                             "bytes_per_token": byts, "achieved_GBs": Bm * byts / (us["median"] * 1e-6) / 1e9,
                             "frac": Bm * byts / (us["median"] * 1e-6) / 1e9 / peak, "tokens_per_s": Bm / (us["median"] * 1e-6)}
    dYs = [torch.randn((Bm, 4, C), device="cuda", generator=g).bfloat16() for _ in range(2)]
    dHm = torch.empty_like(Hm)
    us = timer(lambda i: bk.birkhoff4_backward_mix(Hm, Xs[i % 2], dYs[i % 2], Ys[i % 2], dHm, None, TOL, 20))
    byts = 128 + 3 * 4 * C * 2
    out["fused_mix_backward_bf16"] = {
        "desc": "B=2^16 tokens, C=1024 bf16: dX = P^T dY, G = dY X^T, dH from (P, G), P projected again, one kernel", "us": us,
        "bytes_per_token": byts, "achieved_GBs": Bm * byts / (us["median"] * 1e-6) / 1e9,
        "frac": Bm * byts / (us["median"] * 1e-6) / 1e9 / peak, "tokens_per_s": Bm / (us["median"] * 1e-6)}
    return out


def run_ours(args, wl):
    import torch
    import torch.distributed as dist
    from paper_2606_07574_b200 import binding as bk, inputs, shard

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    bk.lib()                                                                   # raises if libbirkhoff4.so cannot be had
    props = torch.cuda.get_device_properties(local)
    peak, peak_src = measured_peaks()
    B, bf16, max_iter = wl["B"], wl["config"] == 4, wl["max_iter"]
    K, R = args.steps, args.regions

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    clocks = ClockSampler(local)
    clocks.start()
    sm_mhz = clocks.max_mhz or 1965

    # ---- warm-up + the contract's timed region: EXACTLY K steps between two events, barrier + synchronize on both sides
    head, sets, (H0, G0) = None, None, (None, None)
    clocks.region(True)
    head, sets, (H0, G0) = measure_workload(torch, bk, inputs, args.workload, wl, rank, K, R, peak, peak_src, sm_mhz,
                                            props.multi_processor_count)
    nsets = len(sets)
    fwd = bk.birkhoff4_forward_bf16 if bf16 else bk.birkhoff4_forward

    def step(i):
        s, t = sets[i % nsets], sets[(i + 1) % nsets]
        fwd(s["H"], s["P"], TOL, max_iter)
        bk.birkhoff4_backward(t["P"], t["G"], t["dH"])

    for i in range(max(args.warmup, 3)):
        step(i)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    barrier()
    ev[0].record()
    for i in range(K):
        step(i)
    ev[1].record()
    clocks.sample()
    barrier()
    total_ms = shard.reduce_max_time(ev[0].elapsed_time(ev[1]), dist if world > 1 else None)
    value_single = world * B * K / (total_ms * 1e-3)                           # this one region of K steps
    # `value`: the median over the R regions of K steps each (max over ranks of the per-rank median); one region of
    # K = 20 steps is a 1 ms sample
    med_ms = shard.reduce_max_time(head["step_us"]["median"] * 1e-3, dist if world > 1 else None)
    value = world * B / (med_ms * 1e-3)

    # ---- Sinkhorn-20 baseline kernel of the same library (context: PAPER.md:32, 319), fp32 workloads only
    sink = None
    if not bf16:
        us = Timer(torch, min(K, 50), 3)(lambda i: bk.birkhoff4_sinkhorn(sets[i % nsets]["H"], sets[i % nsets]["dH"], 20))
        sink = {"fwd_matrices_per_s": B / (us["median"] * 1e-6), "us": us, **err_stats(torch, sets[0]["dH"])}

    # ---- end to end: pinned host buffers through the host-buffer C-ABI call, copies inside the timed region
    Hh = torch.from_numpy(inputs.bf16_bits_to_f32(H0) if bf16 else H0).pin_memory()
    Gh = torch.from_numpy(G0).pin_memory()
    Ph, dHh = torch.empty_like(Hh).pin_memory(), torch.empty_like(Hh).pin_memory()
    K_e = K if B * K <= (1 << 27) else max(3, (1 << 27) // B)                  # bounded: <= 2^27 matrices end to end
    for _ in range(2):
        bk.birkhoff4_forward_backward_host(Hh, Gh, Ph, dHh, TOL, max_iter)
    barrier()
    t0 = time.perf_counter()
    for _ in range(K_e):
        bk.birkhoff4_forward_backward_host(Hh, Gh, Ph, dHh, TOL, max_iter)     # synchronous: outputs are in host memory
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    clocks.region(False)
    e2e_ms = shard.reduce_max_time(e2e_ms, dist if world > 1 else None)
    e2e = {"value": world * B * K_e / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 2 * B * 64,
           "d2h_bytes_per_step": 2 * B * 64, "steps": K_e,
           "api": "birkhoff4_forward_backward_host(H_host, dP_host -> P_host, dH_host), fp32 pinned host buffers"}
    bk.birkhoff4_host_release()
    del sets, Hh, Gh, Ph, dHh
    torch.cuda.empty_cache()

    if rank != 0:
        clocks.stop()
        if world > 1:
            dist.destroy_process_group()
        return
    fk = head["roofline_kernels"]["forward_kernel"]
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": med_ms, "value_single": value_single, "ms_per_step_single": total_ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "desc": wl["desc"], "B_per_gpu": B, "tol": TOL, "max_iter": max_iter,
                   "parallelism": "batch shards, no collective" if world > 1 else "single GPU",
                   "l2": "rotation over %d buffer sets (>= 1 GiB); backward reads the P written %d steps earlier"
                         % (head["buffer_sets"], head["buffer_sets"] - 1),
                   "repeats": "every per-kernel and per-step time is the median (and min) of %d regions of %d calls" % (R, K)},
        # the dominant kernel is the forward (the Newton solver: the backward is a pure stream); its HBM roofline
        "roofline": dict(fk, kernel="forward_kernel", peak_source=peak_src),
        "roofline_step": head["roofline_step"], "roofline_kernels": head["roofline_kernels"],
        "fwd": {"value": world * head["fwd_matrices_per_s"], "unit": UNIT, "us": head["forward_us"],
                "mean_newton_updates": head["mean_newton_updates"], "update_histogram": head["update_histogram"],
                "unconverged": head["unconverged"]},
        "bwd": {"us": head["backward_us"]}, "step_us": head["step_us"],
        "max_marginal_err": head["max_marginal_err"], "mean_marginal_err": head["mean_marginal_err"],
        "max_err_inf": head["max_err_inf"], "sinkhorn20_gpu": sink, "e2e": e2e,
    }
    if world == 1 and args.workload == "config2" and not args.no_extra:
        clocks.region(True)
        extra = {}
        Kx, Rx = min(K, 20), min(R, 10)
        for name, kw in (("config3_s10", {}), ("config3_s10@max_iter20", {"max_iter": 20}), ("config3_s30", {}),
                         ("config3_s30@max_iter20", {"max_iter": 20}), ("config3_s100", {}),
                         ("config3_s100@max_iter20", {"max_iter": 20}), ("config4", {}), ("config5", {}),
                         ("config5@sorted_by_class", {"sort_by_class": True})):
            base = name.split("@")[0]
            res, s_, _ = measure_workload(torch, bk, inputs, base, WORKLOADS[base], 0, Kx, Rx, peak, peak_src, sm_mhz,
                                          props.multi_processor_count, **kw)
            extra[name] = res
            del s_
            torch.cuda.empty_cache()
        out["workloads"] = extra
        out["widenings"] = measure_widenings(torch, bk, inputs, Kx, min(Rx, 5), peak)
        clocks.region(False)
    clocks.stop()
    out["gpu_launches"] = 2 * K                                               # per timed region of K steps: forward + backward kernel
    out["clocks"] = clocks.summary()
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        n = min(B, 1 << 20 if wl["config"] in (2, 4) else 1 << 14)                # about 10 s of host work
        Hs = inputs.bf16_bits_to_f32(H0[:n]) if bf16 else H0[:n]
        t0 = time.perf_counter()
        oracle_step(oracle, Hs, G0[:n])
        dt = time.perf_counter() - t0
        n1 = max(1024, n // 16)
        t0 = time.perf_counter()
        oracle_step(oracle, Hs[:n1], G0[:n1], nthreads=1)
        dt1 = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": "first %d matrices of buffer set 0, forward+backward, fp64, %.1f s" % (n, dt),
                               "one_thread": {"value": n1 / dt1, "unit": UNIT, "cores": 1,
                                              "sample": "first %d matrices, %.1f s" % (n1, dt1)}}
    out["detail_file"] = write_detail(out)
    sys.stderr.flush()
    print(contract_line(out), flush=True)                                      # the last (and only) stdout line
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--regions", type=int, default=10, help="timed regions of --steps calls per kernel (median and min reported)")
    ap.add_argument("--no-extra", action="store_true", help="config2 only: skip the workloads / widenings blocks")
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    wl = WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_ours(args, wl)


if __name__ == "__main__":
    main()
