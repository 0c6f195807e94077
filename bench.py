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

One JSON line on stdout (rank 0).  `value` = matrices/s through forward+backward with inputs resident in HBM
(K steps between two CUDA events on the launching stream, max over ranks); `e2e` = the same through the
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


def ncu_traffic(kernel, B):
    """dram bytes per launch of `kernel` at batch B from the committed ncu --set full summary, or None"""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            k = [x.strip() for x in line.split(",")]
            if len(k) >= 4 and k[0] == kernel and k[1] == str(B):
                return float(k[2]) + float(k[3])
    return None


def _finite(x):
    """strict JSON: NaN/Inf (e.g. the Sinkhorn-20 baseline's error at s >= 30, where exp underflows) become null"""
    if isinstance(x, float):
        return x if np.isfinite(x) else None
    if isinstance(x, dict):
        return {k: _finite(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_finite(v) for v in x]
    return x


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
    if args.variant:
        bk.birkhoff4_set_variant(args.variant)                                 # measurement only; 0 = library default

    B, bf16, max_iter = wl["B"], wl["config"] == 4, wl["max_iter"]
    set_bytes = B * (32 if bf16 else 64) + 3 * B * 64
    nsets = max(2, -(-(1 << 30) // set_bytes))                                 # >= 1 GiB in rotation
    sets = []
    distinct = 1 if B > (1 << 22) else nsets                                   # 2^24: one draw, copied (host RAM/time)
    for k in range(nsets):
        if k < distinct:
            H, G = make_inputs(wl, rank, k)
            H0, G0 = H, G
        Hd = torch.from_numpy(H.view(np.int16)).cuda().view(torch.bfloat16) if bf16 else torch.from_numpy(H).cuda()
        sets.append(dict(H=Hd, G=torch.from_numpy(G).cuda(), P=torch.empty((B, 4, 4), device="cuda"),
                         dH=torch.empty((B, 4, 4), device="cuda")))
    fwd = bk.birkhoff4_forward_bf16 if bf16 else bk.birkhoff4_forward

    def step(i):
        s, t = sets[i % nsets], sets[(i + 1) % nsets]
        fwd(s["H"], s["P"], TOL, max_iter)
        bk.birkhoff4_backward(t["P"], t["G"], t["dH"])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for s in sets:                                                             # every set has a valid P before backward reads it
        fwd(s["H"], s["P"], TOL, max_iter)
    for i in range(max(args.warmup, 3)):
        step(i)
    clocks = ClockSampler(local)
    clocks.start()

    # ---- device-timed region: K steps, events on the launching (current) stream
    K = args.steps
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
    barrier()
    clocks.region(True)
    ev[0].record()
    for i in range(K):
        step(i)
    ev[1].record()
    clocks.sample()
    barrier()
    total_ms = ev[0].elapsed_time(ev[1])
    # per-kernel average launch duration, same region, same rotation: K launches of one kernel between two events
    ev[2].record()
    for i in range(K):
        s = sets[i % nsets]
        fwd(s["H"], s["P"], TOL, max_iter)
    ev[3].record()
    barrier()
    ev[4].record()
    for i in range(K):
        t = sets[i % nsets]
        bk.birkhoff4_backward(t["P"], t["G"], t["dH"])
    ev[5].record()
    barrier()
    clocks.region(False)
    f_ms, b_ms = ev[2].elapsed_time(ev[3]) / K, ev[4].elapsed_time(ev[5]) / K
    total_ms = shard.reduce_max_time(total_ms, dist if world > 1 else None)
    value = world * B * K / (total_ms * 1e-3)

    # ---- accuracy of what was just computed (set 0), PAPER.md:323 in fp64
    P64 = sets[0]["P"].double()
    err = ((P64.sum(2) - 1).abs().sum(1) + (P64.sum(1) - 1).abs().sum(1))
    max_err, mean_err = float(err.max()), float(err.mean())
    hist = torch.zeros(64, dtype=torch.int64, device="cuda")
    unc = torch.zeros(1, dtype=torch.int64, device="cuda")
    (bk.birkhoff4_forward_bf16_ex if bf16 else bk.birkhoff4_forward_ex)(sets[0]["H"], sets[0]["P"], TOL, max_iter,
                                                                        hist=hist, n_unconverged=unc)
    h = hist.cpu().numpy()
    mean_updates = float((h * np.arange(64)).sum() / max(h.sum(), 1))
    update_hist = {str(k): round(float(h[k]) / max(h.sum(), 1), 6) for k in range(64) if h[k]}
    del P64, err

    # ---- Sinkhorn-20 baseline kernel of the same library (context: PAPER.md:32, 319), fp32 workloads only
    sink = None
    if not bf16:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_s = min(K, 200)
        torch.cuda.synchronize()
        e0.record()
        for i in range(n_s):
            s = sets[i % nsets]
            bk.birkhoff4_sinkhorn(s["H"], s["dH"], 20)
        e1.record()
        torch.cuda.synchronize()
        T64 = sets[(n_s - 1) % nsets]["dH"].double()
        serr = ((T64.sum(2) - 1).abs().sum(1) + (T64.sum(1) - 1).abs().sum(1))
        sink = {"fwd_matrices_per_s": B * n_s / (e0.elapsed_time(e1) * 1e-3), "max_marginal_err": float(serr.max()),
                "mean_marginal_err": float(serr.mean())}
        del T64, serr

    # ---- end to end: pinned host buffers through the host-buffer C-ABI call, copies inside the timed region
    Hh = torch.from_numpy(inputs.bf16_bits_to_f32(H0) if bf16 else H0).pin_memory()
    Gh = torch.from_numpy(G0).pin_memory()
    Ph, dHh = torch.empty_like(Hh).pin_memory(), torch.empty_like(Hh).pin_memory()
    K_e = K if B * K <= (1 << 28) else max(3, (1 << 28) // B)                  # bounded: <= 2^28 matrices end to end
    for _ in range(2):
        bk.birkhoff4_forward_backward_host(Hh, Gh, Ph, dHh, TOL, max_iter)
    barrier()
    clocks.region(True)
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
    clocks.stop()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    fb = 96 if bf16 else FWD_BYTES
    kernels = {
        "forward_lean_kernel": {"bound": "hbm", "achieved": B * fb / (f_ms * 1e-3) / 1e9, "avg_us": f_ms * 1e3,
                           "bytes_per_launch": B * fb},
        "backward_kernel": {"bound": "hbm", "achieved": B * BWD_BYTES / (b_ms * 1e-3) / 1e9, "avg_us": b_ms * 1e3,
                            "bytes_per_launch": B * BWD_BYTES},
    }
    for name, k in kernels.items():
        k.update(peak=peak, unit="GB/s", frac=k["achieved"] / peak, traffic=ncu_traffic(name, B))
    # the forward's second roofline: plain FP32 arithmetic.  Algorithmic work = 150 FP32 thread
    # instructions per evaluation of T, g, Hessian and solve (eqs. (10)-(12)) x (mean updates + 1 final evaluation
    # + 1 for the start-up steps); peak = 128 FP32 lanes per clock per SM at the maximum SM clock.
    props = torch.cuda.get_device_properties(local)
    sm_mhz = clocks.max_mhz or 1965
    alu_peak = 128.0 * props.multi_processor_count * sm_mhz * 1e6 / 1e12
    alu_work = 150.0 * (mean_updates + 2.0)
    alu_ach = B * alu_work / (f_ms * 1e-3) / 1e12
    kernels["forward_lean_kernel"]["alu"] = {
        "bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "T FP32 instr/s", "frac": alu_ach / alu_peak,
        "fp32_instr_per_matrix": alu_work}
    dom = "forward_lean_kernel" if f_ms >= b_ms else "backward_kernel"
    roofline = dict(kernels[dom], kernel=dom, peak_source=peak_src)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "desc": wl["desc"], "B_per_gpu": B, "tol": TOL, "max_iter": max_iter,
                   "variant": args.variant,
                   "parallelism": "batch shards, no collective" if world > 1 else "single GPU",
                   "l2": "rotation over %d buffer sets (%.2f GiB); backward reads the P written %d steps earlier"
                         % (nsets, nsets * set_bytes / 2 ** 30, nsets - 1)},
        "fwd": {"value": world * B / (f_ms * 1e-3), "unit": UNIT, "mean_newton_updates": mean_updates,
                "update_histogram": update_hist,
                "unconverged": int(unc.item())},
        "max_marginal_err": max_err, "mean_marginal_err": mean_err,
        "roofline": roofline, "roofline_kernels": kernels, "sinkhorn20_gpu": sink,
        "e2e": e2e, "gpu_launches": 2 * K, "gpu_launches_per_kernel_timing": 2 * K, "clocks": clocks.summary(),
    }
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        n = min(B, 1 << 20 if wl["config"] in (2, 4) else 1 << 14)                # about 10 s of host work
        Hs = inputs.bf16_bits_to_f32(H0[:n]) if bf16 else H0[:n]
        t0 = time.perf_counter()
        oracle_step(oracle, Hs, G0[:n])
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": "first %d matrices of buffer set 0, forward+backward, fp64, %.1f s" % (n, dt)}
    print(json.dumps(_finite(out)))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--variant", type=int, default=0, help="forward kernel variant (0 = library default)")
    args = ap.parse_args()
    wl = WORKLOADS[args.workload]
    if args.impl == "reference":
        run_reference(args, wl)
    else:
        run_ours(args, wl)


if __name__ == "__main__":
    main()
