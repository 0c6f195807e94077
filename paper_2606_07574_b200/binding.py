"""ctypes binding of libbirkhoff4.so (include/birkhoff4.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  PyTorch supplies device memory and streams
(`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`).  There is NO CPU fallback: calls raise if
the library is missing or a tensor is not on a CUDA device (the *_host calls take CPU tensors by design and
still run on the GPU).
"""
import ctypes
import os

import torch

from . import build as _build

HIST_BINS = 64
_LIB = None


class Birkhoff4Error(RuntimeError):
    pass


def lib():
    """load (building if needed) libbirkhoff4.so; raises if it cannot be had"""
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if not os.path.exists(path) or os.environ.get("BIRKHOFF4_REBUILD"):
            path = _build.build()
        L = ctypes.CDLL(path)
        vp, i64, f32, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_float, ctypes.c_int
        L.birkhoff4_forward.argtypes = [vp, vp, i64, f32, ci, vp]
        L.birkhoff4_forward_ex.argtypes = [vp, vp, i64, f32, ci, vp, vp, vp, vp]
        L.birkhoff4_forward_bf16.argtypes = [vp, vp, i64, f32, ci, vp]
        L.birkhoff4_forward_bf16_ex.argtypes = [vp, vp, i64, f32, ci, vp, vp, vp, vp]
        L.birkhoff4_backward.argtypes = [vp, vp, vp, i64, vp]
        L.birkhoff4_sinkhorn.argtypes = [vp, vp, i64, ci, vp]
        L.birkhoff4_forward_host.argtypes = [vp, vp, i64, f32, ci]
        L.birkhoff4_backward_host.argtypes = [vp, vp, vp, i64]
        L.birkhoff4_forward_backward_host.argtypes = [vp, vp, vp, vp, i64, f32, ci]
        L.birkhoff4_host_release.argtypes = []
        L.birkhoff4_host_release.restype = None
        L.birkhoff4_set_variant.argtypes = [ci]
        L.birkhoff4_strerror.argtypes = [ci]
        L.birkhoff4_strerror.restype = ctypes.c_char_p
        L.birkhoff4_version.argtypes = []
        for name in ("forward", "forward_ex", "forward_bf16", "forward_bf16_ex", "backward", "sinkhorn", "forward_host",
                     "backward_host", "forward_backward_host", "set_variant", "version"):
            getattr(L, "birkhoff4_" + name).restype = ci
        _LIB = L
    return _LIB


def _check(rc):
    if rc != 0:
        raise Birkhoff4Error("birkhoff4 error %d: %s" % (rc, lib().birkhoff4_strerror(rc).decode()))


def _dev(t, dtype, name):
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise Birkhoff4Error("%s must be a CUDA tensor (there is no CPU path)" % name)
    if t.dtype != dtype or not t.is_contiguous() or t.numel() % 16:
        raise Birkhoff4Error("%s must be a contiguous %s tensor of [B,4,4]" % (name, dtype))
    return t


def _host(t, name):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.numel() % 16:
        raise Birkhoff4Error("%s must be a contiguous float32 CPU tensor of [B,4,4]" % name)
    return t


def _stream(stream):
    return ctypes.c_void_p((stream if stream is not None else torch.cuda.current_stream()).cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr() if t is not None else 0)


def birkhoff4_forward(H, P=None, tol=1e-6, max_iter=20, stream=None):
    """P = proj^KL(exp(H)) for fp32 CUDA H[B,4,4]; asynchronous on `stream` (default: current stream)."""
    H = _dev(H, torch.float32, "H")
    P = torch.empty_like(H) if P is None else _dev(P, torch.float32, "P")
    _check(lib().birkhoff4_forward(_ptr(H), _ptr(P), H.numel() // 16, tol, max_iter, _stream(stream)))
    return P


def _diag_check(B, iters, hist, n_unconverged):
    if iters is not None and (iters.dtype != torch.int32 or iters.numel() != B or not iters.is_cuda):
        raise Birkhoff4Error("iters must be a CUDA int32 tensor of [B]")
    if hist is not None and (hist.dtype != torch.int64 or hist.numel() != HIST_BINS or not hist.is_cuda):
        raise Birkhoff4Error("hist must be a CUDA int64 tensor of [64]")
    if n_unconverged is not None and (n_unconverged.dtype != torch.int64 or n_unconverged.numel() != 1
                                      or not n_unconverged.is_cuda):
        raise Birkhoff4Error("n_unconverged must be a CUDA int64 tensor of [1]")


def birkhoff4_forward_ex(H, P=None, tol=1e-6, max_iter=20, iters=None, hist=None, n_unconverged=None, stream=None):
    """forward + diagnostics; iters int32[B], hist int64[64] (accumulated), n_unconverged int64[1] (accumulated)"""
    H = _dev(H, torch.float32, "H")
    P = torch.empty_like(H) if P is None else _dev(P, torch.float32, "P")
    B = H.numel() // 16
    _diag_check(B, iters, hist, n_unconverged)
    _check(lib().birkhoff4_forward_ex(_ptr(H), _ptr(P), B, tol, max_iter, _ptr(iters), _ptr(hist),
                                      _ptr(n_unconverged), _stream(stream)))
    return P


def birkhoff4_forward_bf16(H, P=None, tol=1e-6, max_iter=20, stream=None):
    """forward for bf16 logits (torch.bfloat16 CUDA tensor [B,4,4]); P is fp32"""
    H = _dev(H, torch.bfloat16, "H")
    P = torch.empty(H.shape, dtype=torch.float32, device=H.device) if P is None else _dev(P, torch.float32, "P")
    _check(lib().birkhoff4_forward_bf16(_ptr(H), _ptr(P), H.numel() // 16, tol, max_iter, _stream(stream)))
    return P


def birkhoff4_forward_bf16_ex(H, P=None, tol=1e-6, max_iter=20, iters=None, hist=None, n_unconverged=None, stream=None):
    """bf16-logit forward + the diagnostics of birkhoff4_forward_ex"""
    H = _dev(H, torch.bfloat16, "H")
    P = torch.empty(H.shape, dtype=torch.float32, device=H.device) if P is None else _dev(P, torch.float32, "P")
    B = H.numel() // 16
    _diag_check(B, iters, hist, n_unconverged)
    _check(lib().birkhoff4_forward_bf16_ex(_ptr(H), _ptr(P), B, tol, max_iter, _ptr(iters), _ptr(hist),
                                           _ptr(n_unconverged), _stream(stream)))
    return P


def birkhoff4_backward(P, dP, dH=None, stream=None):
    """dH = dL/dH from the forward output P and dP = dL/dP (fp32 CUDA [B,4,4])"""
    P = _dev(P, torch.float32, "P")
    dP = _dev(dP, torch.float32, "dP")
    if dP.numel() != P.numel():
        raise Birkhoff4Error("P and dP must have the same shape")
    dH = torch.empty_like(P) if dH is None else _dev(dH, torch.float32, "dH")
    _check(lib().birkhoff4_backward(_ptr(P), _ptr(dP), _ptr(dH), P.numel() // 16, _stream(stream)))
    return dH


def birkhoff4_sinkhorn(H, P=None, n_iter=20, stream=None):
    """Sinkhorn-Knopp baseline: n_iter x (row normalise, column normalise) of exp(H)"""
    H = _dev(H, torch.float32, "H")
    P = torch.empty_like(H) if P is None else _dev(P, torch.float32, "P")
    _check(lib().birkhoff4_sinkhorn(_ptr(H), _ptr(P), H.numel() // 16, n_iter, _stream(stream)))
    return P


def birkhoff4_forward_host(H_host, P_host=None, tol=1e-6, max_iter=20):
    """host-buffer forward: CPU tensors in and out (pinned recommended), copies + kernel inside; synchronous"""
    H_host = _host(H_host, "H_host")
    P_host = torch.empty_like(H_host) if P_host is None else _host(P_host, "P_host")
    _check(lib().birkhoff4_forward_host(_ptr(H_host), _ptr(P_host), H_host.numel() // 16, tol, max_iter))
    return P_host


def birkhoff4_backward_host(P_host, dP_host, dH_host=None):
    P_host = _host(P_host, "P_host")
    dP_host = _host(dP_host, "dP_host")
    dH_host = torch.empty_like(P_host) if dH_host is None else _host(dH_host, "dH_host")
    _check(lib().birkhoff4_backward_host(_ptr(P_host), _ptr(dP_host), _ptr(dH_host), P_host.numel() // 16))
    return dH_host


def birkhoff4_forward_backward_host(H_host, dP_host, P_host=None, dH_host=None, tol=1e-6, max_iter=20, want_P=True):
    """host-buffer forward + backward; P stays on the device between the two kernels"""
    H_host = _host(H_host, "H_host")
    dP_host = _host(dP_host, "dP_host")
    if want_P and P_host is None:
        P_host = torch.empty_like(H_host)
    dH_host = torch.empty_like(H_host) if dH_host is None else _host(dH_host, "dH_host")
    _check(lib().birkhoff4_forward_backward_host(_ptr(H_host), _ptr(dP_host), _ptr(P_host), _ptr(dH_host),
                                                 H_host.numel() // 16, tol, max_iter))
    return P_host, dH_host


def birkhoff4_host_release():
    lib().birkhoff4_host_release()


def birkhoff4_set_variant(variant):
    """0 = default (4); 1/2 = guarded solver for every matrix, one/two matrices per thread; 3/4 = lean iteration
    for well-scaled logits + guarded solver for the rest, 3/4 blocks per SM (include/birkhoff4.h)"""
    return lib().birkhoff4_set_variant(int(variant))


def birkhoff4_version():
    return lib().birkhoff4_version()
