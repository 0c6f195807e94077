"""birkhoff4_forward_host_static: the host-buffer forward for callers that cannot allocate device memory.

Some processes cannot call cudaMalloc when they need a projection: the GPU's memory has all been claimed by the
process's own pool (an inference server's KV cache, a training job's caching allocator), a device-wide stall is
not acceptable, or another thread is recording a CUDA graph.  For them the library keeps the device copy of the
batch in a fixed 4 MiB array of its own (BIRKHOFF4_STATIC_MAX = 65536 matrices) instead of in buffers it allocates.

What is checked: the new call returns what the existing device-pointer forward returns for the same logits (the same
kernel runs, so the results should be identical; the gate is the suite's forward tolerance, max |dP| <= 1e-5), on two
calls in a row that reuse the array -- the second one shorter and with different logits, so that matrices left
behind by the first call sit in the array beyond its end -- and that a batch over the limit is refused with a
message that names the limit.  The file sorts last on purpose: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It depends on no other test and on no state they leave.
"""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")
from paper_2606_07574_b200 import binding as bk, inputs

TOL_P = 1e-5            # the forward gate of tests/test_gpu_parity.py


def test_over_the_limit_is_refused_before_the_device_is_touched():
    """B > BIRKHOFF4_STATIC_MAX: a clear error and no copy or launch (so this runs without a GPU too)"""
    L = bk.lib()
    rc = L.birkhoff4_forward_host_static(ctypes.c_void_p(64), ctypes.c_void_p(64), bk.STATIC_MAX + 1, 1e-6, 20, None)
    assert rc == 2
    msg = L.birkhoff4_strerror(rc).decode()
    assert "65536" in msg and "too large" in msg
    assert L.birkhoff4_forward_host_static(None, None, 0, 1e-6, 20, None) == 0       # B == 0: no-op
    assert L.birkhoff4_forward_host_static(None, None, -1, 1e-6, 20, None) == 1
    assert L.birkhoff4_forward_host_static(None, None, 8, 1e-6, 20, None) == 1       # null host pointers
    assert L.birkhoff4_forward_host_static(ctypes.c_void_p(64), ctypes.c_void_p(64), 8, -1.0, 20, None) == 1
    with pytest.raises(bk.Birkhoff4Error, match="65536"):
        bk.birkhoff4_forward_host_static(torch.zeros(bk.STATIC_MAX + 1, 4, 4))


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_device_pointer_forward():
    first = inputs.normal(bk.STATIC_MAX, 1.0, config=71)[0]        # the largest batch the call takes
    second = inputs.normal(1000, 10.0, config=72)[0]               # shorter, ragged, wide logits
    for H in (first, second):
        H_host = torch.from_numpy(np.ascontiguousarray(H))
        want = bk.birkhoff4_forward(H_host.cuda(), tol=1e-6, max_iter=20)          # the existing path
        torch.cuda.synchronize()
        want = want.cpu().numpy()
        got = bk.birkhoff4_forward_host_static(H_host, tol=1e-6, max_iter=20).numpy()
        assert got.shape == H.shape and np.isfinite(got).all()
        assert np.abs(got - want).max() <= TOL_P
        assert np.abs(got.sum(1) - 1).max() <= 1e-6 and np.abs(got.sum(2) - 1).max() <= 1e-6
    # pinned buffers, the output written over the input, a stream of the caller's
    H_pin = torch.from_numpy(np.ascontiguousarray(second)).pin_memory()
    st = torch.cuda.Stream()
    out = bk.birkhoff4_forward_host_static(H_pin, H_pin, stream=st)
    assert out is H_pin and np.abs(out.numpy() - want).max() <= TOL_P
