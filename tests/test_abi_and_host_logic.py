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
