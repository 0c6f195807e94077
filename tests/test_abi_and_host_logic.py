"""CPU-only checks of the boundary and the host logic: libbirkhoff4.so builds (nvcc cross-compiles for sm_100a
without a GPU), loads, and exports every symbol include/birkhoff4.h declares; argument validation that needs no
device; the binding refuses CPU tensors (no CPU fallback); batch sharding for N > 1 ranks, exercised with a
world_size-2 gloo group.  No compute call is made here."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "birkhoff4.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2606_07574_b200 import build
    return ctypes.CDLL(build.build())


HEADERS = sorted(os.path.join(ROOT, "include", f) for f in os.listdir(os.path.join(ROOT, "include")) if f.endswith(".h"))


def declared_symbols():
    """every function declared in include/*.h"""
    names = set()
    for h in HEADERS:
        src = re.sub(r"/\*.*?\*/", "", open(h).read(), flags=re.S)
        names |= set(re.findall(r"\b((?:birkhoff[0-9]*|entropic_ot|birkhoff_mix)_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text("".join('#include "%s"\n' % os.path.basename(h) for h in HEADERS) + "int main(void) { return BIRKHOFF4_OK; }\n")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert {"birkhoff4_forward", "birkhoff4_backward", "birkhoff4_forward_ex", "birkhoff4_forward_bf16",
            "birkhoff4_sinkhorn", "birkhoff4_forward_backward_host", "birkhoff4_strerror",
            "birkhoff4_version", "birkhoff4_forward_backward", "birkhoff4_forward_guarded", "birkhoff8_forward",
            "birkhoff8_backward", "entropic_ot_forward", "entropic_ot_backward"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "missing export " + n


def test_library_has_no_torch_or_oracle_dependency():
    from paper_2606_07574_b200 import build
    out = subprocess.run(["ldd", build.LIB], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out and "libcudart" not in out      # cudart is linked statically


def test_library_is_sm100a_sass():
    from paper_2606_07574_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_version_strerror_and_validation_without_device(lib):
    lib.birkhoff4_strerror.restype = ctypes.c_char_p
    assert lib.birkhoff4_version() >= 100
    assert lib.birkhoff4_strerror(0) == b"success"
    assert b"invalid" in lib.birkhoff4_strerror(1)
    vp, i64, f32, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_float, ctypes.c_int
    lib.birkhoff4_forward.argtypes = [vp, vp, i64, f32, ci, vp]
    lib.birkhoff4_backward.argtypes = [vp, vp, vp, i64, vp]
    lib.birkhoff4_sinkhorn.argtypes = [vp, vp, i64, ci, vp]
    assert lib.birkhoff4_forward(None, None, 0, 1e-6, 20, None) == 0                 # B == 0: no-op
    assert lib.birkhoff4_forward(None, None, -1, 1e-6, 20, None) == 1
    assert lib.birkhoff4_forward(None, None, 8, 1e-6, 20, None) == 1                 # null pointers
    assert lib.birkhoff4_forward(64, 64, 8, -1.0, 20, None) == 1
    assert lib.birkhoff4_forward(64, 64, 8, float("nan"), 20, None) == 1
    assert lib.birkhoff4_forward(64, 64, 8, 1e-6, -3, None) == 1
    assert lib.birkhoff4_forward(68, 64, 8, 1e-6, 20, None) == 1                     # misaligned
    assert lib.birkhoff4_backward(64, None, 64, 8, None) == 1
    assert lib.birkhoff4_backward(None, None, None, 0, None) == 0
    assert lib.birkhoff4_sinkhorn(64, 64, 8, -1, None) == 1


def test_binding_refuses_cpu_tensors():
    torch = pytest.importorskip("torch")
    from paper_2606_07574_b200 import binding as bk
    x = torch.zeros(4, 4, 4)
    for call in (lambda: bk.birkhoff4_forward(x), lambda: bk.birkhoff4_backward(x, x), lambda: bk.birkhoff4_sinkhorn(x),
                 lambda: bk.birkhoff4_forward_bf16(x.bfloat16())):
        with pytest.raises(bk.Birkhoff4Error):
            call()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_07574_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "birkhoff4_oracle" not in src and "bk4o_" not in src, f


def test_inputs_are_seeded_and_structured():
    from paper_2606_07574_b200 import inputs
    a, b = inputs.make(1), inputs.make(1)
    assert np.array_equal(a["H"], b["H"]) and np.array_equal(a["G"], b["G"])
    assert a["H"].shape == (1024, 4, 4) and a["H"].dtype == np.float32
    c4 = inputs.make(4, B=4096)
    assert c4["H"].dtype == np.uint16 and np.array_equal(inputs.f32_to_bf16_bits(c4["H_f32"]), c4["H"])
    assert abs(c4["H_f32"].std() - 2.0) < 0.05
    c5 = inputs.make(5, B=1 << 15)
    frac = np.bincount(c5["cls"], minlength=4) / float(1 << 15)
    assert np.abs(frac - [0.5, 0.25, 0.125, 0.125]).max() < 0.02
    dup = c5["H"][c5["cls"] == 2]
    assert all(any(np.array_equal(m[i], m[j]) for i in range(4) for j in range(i)) for m in dup[:200])
    ties = np.sort(c5["H"][c5["cls"] == 3], axis=2)
    assert np.array_equal(ties[:, :, 3], ties[:, :, 2])
    s3 = inputs.make(3, B=1 << 14, s=30.0)
    assert abs(s3["H"].std() / 30.0 - 1) < 0.02


def test_shard_bounds_cover_the_batch():
    from paper_2606_07574_b200 import shard
    for B in (0, 1, 7, 1 << 20, (1 << 20) + 3):
        for w in (1, 2, 3, 8):
            cuts = [shard.shard_bounds(B, w, r) for r in range(w)]
            assert cuts[0][0] == 0 and cuts[-1][1] == B
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(w - 1))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_bounds(10, 2, 2)


_WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
from paper_2606_07574_b200 import shard
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
lo, hi = shard.shard_bounds(1001, w, r)
t = shard.reduce_max_time(10.0 + 5.0 * r, dist)
assert t == 15.0, t
print("rank %d shard %d %d max %.1f" % (r, lo, hi, t))
dist.destroy_process_group()
"""


def test_two_rank_gloo_sharding_and_timing(tmp_path):
    pytest.importorskip("torch")
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    port = 29500 + os.getpid() % 2000
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(w), ROOT],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "rank 0 shard 0 501 max 15.0" in out.stdout and "rank 1 shard 501 1001 max 15.0" in out.stdout


def test_bench_reference_arm_runs_on_cpu():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2",
                          "--warmup", "1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "matrices/s"
    assert len(out.stdout.strip().splitlines()[-1]) < 2048


def _canned_bench_result():
    """a full bench result of the shape run_ours() builds, with made-up numbers (no GPU): what contract_line() is fed"""
    us = {"median": 28.123456789, "min": 27.987654321, "regions": 10, "calls_per_region": 20}
    kern = lambda frac: {"bound": "hbm", "achieved": 4673.123456, "peak": 6556.8, "unit": "GB/s", "frac": frac,   # noqa: E731
                         "frac_min_time": 0.72, "frac_of_nominal_7700": 0.61, "avg_us": 28.123456789, "min_us": 27.9,
                         "bytes_per_launch": 134217728, "traffic": 91435776.0, "isolated_us": 31.4, "frac_isolated": 0.652,
                         "issue_diagnostic": {"bound": "alu", "frac": 0.5, "peak_source": "x" * 300},
                         "work_roofline": {"bound": "fp32", "frac": 0.74, "floor_us": 20.6, "peak_source": "y" * 200}}
    wl = {"desc": "B=2^20 fp32, H iid N(0,10^2)", "step_us": us, "forward_us": us, "backward_us": us, "max_marginal_err": 9.6e-7,
          "roofline_kernels": {"forward_kernel": kern(0.48), "backward_kernel": kern(1.01)},
          "update_histogram": {str(k): 0.01 for k in range(40)}}
    names = ["config3_s10", "config3_s10@max_iter20", "config3_s30", "config3_s30@max_iter20", "config3_s100",
             "config3_s100@max_iter20", "config4", "config5", "config5@sorted_by_class"]
    return {
        "metric": "4x4 projections/sec fwd+bwd", "value": 1.8234567891e10, "unit": "matrices/s", "n_gpus": 1, "steps": 20,
        "warmup": 5, "ms_per_step": 0.0573123456, "value_single": 1.81e10, "ms_per_step_single": 0.0579,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "config2", "desc": "B=2^20 fp32, H,dP iid N(0,1)", "B_per_gpu": 1 << 20, "tol": 1e-6,
                   "max_iter": 20, "parallelism": "single GPU",
                   "l2": "rotation over 5 buffer sets (>= 1 GiB); backward reads the P written 4 steps earlier",
                   "repeats": "every per-kernel and per-step time is the median (and min) of 10 regions of 20 calls"},
        "roofline": dict(kern(0.713), kernel="forward_kernel", peak_source="measured (MEASURED_PEAKS.json hbm_gbs)"),
        "roofline_step": {"bound": "hbm", "achieved": 5855.1, "peak": 6556.8, "unit": "GB/s", "frac": 0.893,
                          "bytes_per_step": 335544320, "peak_source": "measured (MEASURED_PEAKS.json hbm_gbs)"},
        "roofline_kernels": {"forward_kernel": kern(0.713), "backward_kernel": kern(1.01)},
        "fwd": {"value": 3.7e10, "unit": "matrices/s", "us": us, "mean_newton_updates": 2.31,
                "update_histogram": {"2": 0.7, "3": 0.29, "4": 0.01}, "unconverged": 0},
        "bwd": {"us": us}, "step_us": us, "max_marginal_err": 9.5e-7, "mean_marginal_err": 2.2e-7, "max_err_inf": 2.4e-7,
        "sinkhorn20_gpu": {"fwd_matrices_per_s": 4e10, "us": us, "max_marginal_err": float("nan")},
        "e2e": {"value": 3.18e8, "unit": "matrices/s", "h2d_bytes_per_step": 1 << 27, "d2h_bytes_per_step": 1 << 27, "steps": 20,
                "api": "birkhoff4_forward_backward_host(H_host, dP_host -> P_host, dH_host), fp32 pinned host buffers"},
        "workloads": {n: wl for n in names}, "widenings": {"x": {"us": us}},
        "gpu_launches": 5440, "gpu_launches_timed_region": 40,
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965, "reasons": ["sw_power_cap"], "samples": 812},
        "cpu_baseline": {"value": 1.1e5, "unit": "matrices/s", "cores": 32, "kind": "oracle",
                         "sample": "first 1048576 matrices of buffer set 0, forward+backward, fp64, 9.8 s",
                         "one_thread": {"value": 5e3, "unit": "matrices/s", "cores": 1, "sample": "first 65536 matrices, 12.9 s"}},
        "detail_file": "gpurun_out/bench_detail.json",
    }


def test_bench_contract_line_is_compact_and_complete():
    """the one stdout line of bench.py: strict JSON, under 2 KB, every key of the driver's contract present (round 2's
    26 KB line could not be parsed from the driver's bounded stdout tail)"""
    import json
    sys.path.insert(0, ROOT)
    import bench
    text = bench.contract_line(_canned_bench_result())
    assert len(text) < bench.LINE_LIMIT == 2048 and "\n" not in text and "NaN" not in text
    line = json.loads(text)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert k in line, k
    assert line["value"] > 0 and line["config"]["workload"] == "config2"
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(line["roofline"])
    assert line["roofline"]["bound"] == "hbm" and abs(line["roofline"]["frac"] - 0.713) < 1e-3
    assert {"value", "unit", "cores", "kind", "sample"} == set(line["cpu_baseline"])
    assert {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} <= set(line["e2e"])
    assert sorted(line["per_config"]) == ["config3_s10", "config3_s100", "config3_s30", "config4", "config5"]
    assert len(line["per_config"]["config5"]) == 5
    assert line["roofline"]["work_bound"] == "fp32" and abs(line["roofline"]["work_frac"] - 0.74) < 1e-3
