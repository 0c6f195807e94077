"""ctypes binding of libbirkhoff4.so (include/birkhoff4.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  PyTorch supplies device memory and streams
(`tensor.data_ptr()`, `torch.cuda.current_stream(device).cuda_stream`).  There is NO CPU fallback: calls raise if
the library is missing or a tensor is not on a CUDA device (the *_host calls take CPU tensors by design and still
run on the GPU).

What the marshalling checks before a raw pointer reaches the library: dtype, contiguity, element count of every
tensor against the batch size taken from the first one, all tensors on one CUDA device; the call is made with that
device current and on that device's current stream unless a stream is passed.
"""
import ctypes
import os

import torch

from . import build as _build

HIST_BINS = 64
STATIC_MAX = 65536      # BIRKHOFF4_STATIC_MAX: matrices per call of birkhoff4_forward_host_static
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
        sig = {
            "forward": [vp, vp, i64, f32, ci, vp],
            "forward_ex": [vp, vp, i64, f32, ci, vp, vp, vp, vp],
            "forward_guarded": [vp, vp, i64, f32, ci, vp, vp, vp, vp],
            "forward_bf16": [vp, vp, i64, f32, ci, vp],
            "forward_bf16_ex": [vp, vp, i64, f32, ci, vp, vp, vp, vp],
            "backward": [vp, vp, vp, i64, vp],
            "forward_backward": [vp, vp, vp, vp, i64, f32, ci, vp],
            "forward_mix": [vp, vp, vp, vp, i64, ci, f32, ci, vp],
            "forward_mix_bf16": [vp, vp, vp, vp, i64, ci, f32, ci, vp],
            "backward_mix": [vp, vp, vp, vp, vp, vp, i64, ci, f32, ci, vp],
            "backward_mix_bf16": [vp, vp, vp, vp, vp, vp, i64, ci, f32, ci, vp],
            "sinkhorn": [vp, vp, i64, ci, vp],
            "forward_host": [vp, vp, i64, f32, ci],
            "backward_host": [vp, vp, vp, i64],
            "forward_backward_host": [vp, vp, vp, vp, i64, f32, ci],
            "forward_host_static": [vp, vp, i64, f32, ci, vp],
            "version": [],
        }
        for name, args in sig.items():
            f = getattr(L, "birkhoff4_" + name)
            f.argtypes, f.restype = args, ci
        L.birkhoff8_forward.argtypes, L.birkhoff8_forward.restype = [vp, vp, i64, f32, ci, vp, vp, vp], ci
        L.birkhoff8_backward.argtypes, L.birkhoff8_backward.restype = [vp, vp, vp, i64, vp], ci
        L.entropic_ot_forward.argtypes = [vp, vp, vp, vp, i64, ci, ci, f32, f32, ci, vp, vp, vp]
        L.entropic_ot_forward.restype = ci
        L.entropic_ot_backward.argtypes, L.entropic_ot_backward.restype = [vp, vp, vp, i64, ci, ci, f32, vp], ci
        L.birkhoff4_host_release.argtypes = []
        L.birkhoff4_host_release.restype = None
        L.birkhoff4_strerror.argtypes = [ci]
        L.birkhoff4_strerror.restype = ctypes.c_char_p
        _LIB = L
    return _LIB


def _check(rc):
    if rc != 0:
        raise Birkhoff4Error("birkhoff4 error %d: %s" % (rc, lib().birkhoff4_strerror(rc).decode()))


def _dev(t, dtype, name, numel=None, like=None):
    """a contiguous CUDA tensor of `dtype` with `numel` elements (if given) on the device of `like` (if given)"""
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise Birkhoff4Error("%s must be a CUDA tensor (there is no CPU path)" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise Birkhoff4Error("%s must be a contiguous %s tensor" % (name, dtype))
    if numel is not None and t.numel() != numel:
        raise Birkhoff4Error("%s has %d elements, expected %d" % (name, t.numel(), numel))
    if like is not None and t.device != like.device:
        raise Birkhoff4Error("%s is on %s, expected %s" % (name, t.device, like.device))
    return t


def _batch(t, per, name):
    if t.numel() % per:
        raise Birkhoff4Error("%s must hold whole matrices of %d elements" % (name, per))
    return t.numel() // per


def _host(t, name, numel=None):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.numel() % 16:
        raise Birkhoff4Error("%s must be a contiguous float32 CPU tensor of [B,4,4]" % name)
    if numel is not None and t.numel() != numel:
        raise Birkhoff4Error("%s has %d elements, expected %d" % (name, t.numel(), numel))
    return t


def _stream(stream, device):
    return ctypes.c_void_p((stream if stream is not None else torch.cuda.current_stream(device)).cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr() if t is not None else 0)


def _out(P, like, name, dtype=torch.float32):
    if P is None:
        return torch.empty(like.shape, dtype=dtype, device=like.device)
    return _dev(P, dtype, name, like.numel(), like)


def _diag_check(B, like, iters, hist, n_unconverged):
    if iters is not None:
        _dev(iters, torch.int32, "iters", B, like)
    if hist is not None:
        _dev(hist, torch.int64, "hist", HIST_BINS, like)
    if n_unconverged is not None:
        _dev(n_unconverged, torch.int64, "n_unconverged", 1, like)


def birkhoff4_forward(H, P=None, tol=1e-6, max_iter=20, stream=None):
    """P = proj^KL(exp(H)) for fp32 CUDA H[B,4,4]; asynchronous on `stream` (default: current stream)."""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 16, "H")
    P = _out(P, H, "P")
    with torch.cuda.device(H.device):
        _check(lib().birkhoff4_forward(_ptr(H), _ptr(P), B, tol, max_iter, _stream(stream, H.device)))
    return P


def _forward_diag(fn, H, dtype, P, tol, max_iter, iters, hist, n_unconverged, stream):
    H = _dev(H, dtype, "H")
    B = _batch(H, 16, "H")
    P = _out(P, H, "P")
    _diag_check(B, H, iters, hist, n_unconverged)
    with torch.cuda.device(H.device):
        _check(fn(_ptr(H), _ptr(P), B, tol, max_iter, _ptr(iters), _ptr(hist), _ptr(n_unconverged),
                  _stream(stream, H.device)))
    return P


def birkhoff4_forward_ex(H, P=None, tol=1e-6, max_iter=20, iters=None, hist=None, n_unconverged=None, stream=None):
    """forward + diagnostics; iters int32[B], hist int64[64] (accumulated), n_unconverged int64[1] (accumulated)"""
    return _forward_diag(lib().birkhoff4_forward_ex, H, torch.float32, P, tol, max_iter, iters, hist, n_unconverged, stream)


def birkhoff4_forward_guarded(H, P=None, tol=1e-6, max_iter=20, iters=None, hist=None, n_unconverged=None, stream=None):
    """the guarded solver for every matrix (validation of the default path); diagnostics as in birkhoff4_forward_ex"""
    return _forward_diag(lib().birkhoff4_forward_guarded, H, torch.float32, P, tol, max_iter, iters, hist, n_unconverged,
                         stream)


def birkhoff4_forward_bf16(H, P=None, tol=1e-6, max_iter=20, stream=None):
    """forward for bf16 logits (torch.bfloat16 CUDA tensor [B,4,4]); P is fp32"""
    H = _dev(H, torch.bfloat16, "H")
    B = _batch(H, 16, "H")
    P = _out(P, H, "P")
    with torch.cuda.device(H.device):
        _check(lib().birkhoff4_forward_bf16(_ptr(H), _ptr(P), B, tol, max_iter, _stream(stream, H.device)))
    return P


def birkhoff4_forward_bf16_ex(H, P=None, tol=1e-6, max_iter=20, iters=None, hist=None, n_unconverged=None, stream=None):
    """bf16-logit forward + the diagnostics of birkhoff4_forward_ex"""
    return _forward_diag(lib().birkhoff4_forward_bf16_ex, H, torch.bfloat16, P, tol, max_iter, iters, hist, n_unconverged,
                         stream)


def birkhoff4_backward(P, dP, dH=None, stream=None):
    """dH = dL/dH from the forward output P and dP = dL/dP (fp32 CUDA [B,4,4])"""
    P = _dev(P, torch.float32, "P")
    B = _batch(P, 16, "P")
    dP = _dev(dP, torch.float32, "dP", P.numel(), P)
    dH = _out(dH, P, "dH")
    with torch.cuda.device(P.device):
        _check(lib().birkhoff4_backward(_ptr(P), _ptr(dP), _ptr(dH), B, _stream(stream, P.device)))
    return dH


def birkhoff4_forward_backward(H, dP, P=None, dH=None, tol=1e-6, max_iter=20, want_P=True, stream=None):
    """fused forward + backward (one kernel): returns (P or None, dH); P is not written when want_P is False"""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 16, "H")
    dP = _dev(dP, torch.float32, "dP", H.numel(), H)
    if want_P or P is not None:
        P = _out(P, H, "P")
    dH = _out(dH, H, "dH")
    with torch.cuda.device(H.device):
        _check(lib().birkhoff4_forward_backward(_ptr(H), _ptr(dP), _ptr(P), _ptr(dH), B, tol, max_iter,
                                                _stream(stream, H.device)))
    return P, dH


def birkhoff4_forward_mix(H, X, Y=None, P=None, tol=1e-6, max_iter=20, want_P=False, stream=None):
    """fused consumer: Y[b] = proj(exp(H[b])) @ X[b] for X[B,4,C] (fp32 or bfloat16 CUDA); returns (Y, P or None)"""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 16, "H")
    if not isinstance(X, torch.Tensor) or X.dtype not in (torch.float32, torch.bfloat16):
        raise Birkhoff4Error("X must be a float32 or bfloat16 tensor")
    X = _dev(X, X.dtype, "X", like=H)
    if X.dim() != 3 or X.shape[0] != B or X.shape[1] != 4:
        raise Birkhoff4Error("X must be [B,4,C]")
    C = X.shape[2]
    Y = _out(Y, X, "Y", X.dtype)
    if want_P or P is not None:
        P = _out(P, H, "P")
    fn = lib().birkhoff4_forward_mix if X.dtype == torch.float32 else lib().birkhoff4_forward_mix_bf16
    with torch.cuda.device(H.device):
        _check(fn(_ptr(H), _ptr(X), _ptr(Y), _ptr(P), B, C, tol, max_iter, _stream(stream, H.device)))
    return Y, P


def birkhoff4_backward_mix(H, X, dY, dX=None, dH=None, P=None, tol=1e-6, max_iter=20, want_P=False, stream=None):
    """backward of the fused consumer in one kernel: dX[b] = P[b]^T dY[b] and dH[b] = dL/dH[b] from G[b] = dY[b] X[b]^T, with
    P[b] = proj(exp(H[b])) projected again from the logits; X, dY [B,4,C] fp32 or bfloat16 CUDA.  Returns (dX, dH, P or None)"""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 16, "H")
    if not isinstance(X, torch.Tensor) or X.dtype not in (torch.float32, torch.bfloat16):
        raise Birkhoff4Error("X must be a float32 or bfloat16 tensor")
    X = _dev(X, X.dtype, "X", like=H)
    if X.dim() != 3 or X.shape[0] != B or X.shape[1] != 4:
        raise Birkhoff4Error("X must be [B,4,C]")
    C = X.shape[2]
    dY = _dev(dY, X.dtype, "dY", X.numel(), H)
    dX = _out(dX, X, "dX", X.dtype)
    dH = _out(dH, H, "dH")
    if want_P or P is not None:
        P = _out(P, H, "P")
    fn = lib().birkhoff4_backward_mix if X.dtype == torch.float32 else lib().birkhoff4_backward_mix_bf16
    with torch.cuda.device(H.device):
        _check(fn(_ptr(H), _ptr(X), _ptr(dY), _ptr(dX), _ptr(dH), _ptr(P), B, C, tol, max_iter, _stream(stream, H.device)))
    return dX, dH, P


def birkhoff4_sinkhorn(H, P=None, n_iter=20, stream=None):
    """Sinkhorn-Knopp baseline: n_iter x (row normalise, column normalise) of exp(H)"""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 16, "H")
    P = _out(P, H, "P")
    with torch.cuda.device(H.device):
        _check(lib().birkhoff4_sinkhorn(_ptr(H), _ptr(P), B, n_iter, _stream(stream, H.device)))
    return P


def birkhoff4_forward_host(H_host, P_host=None, tol=1e-6, max_iter=20):
    """host-buffer forward: CPU tensors in and out (pinned recommended), copies + kernel inside; synchronous"""
    H_host = _host(H_host, "H_host")
    P_host = torch.empty_like(H_host) if P_host is None else _host(P_host, "P_host", H_host.numel())
    _check(lib().birkhoff4_forward_host(_ptr(H_host), _ptr(P_host), H_host.numel() // 16, tol, max_iter))
    return P_host


def birkhoff4_forward_host_static(H_host, P_host=None, tol=1e-6, max_iter=20, stream=None):
    """birkhoff4_forward_host without any device allocation, for at most STATIC_MAX (65536) matrices per call.

    For processes in which cudaMalloc is not an option: all GPU memory already belongs to the process's own pool
    (a serving engine's KV cache, a grown caching allocator), a device-wide stall cannot be afforded, or another
    thread is capturing a CUDA graph.  The device copy of the batch sits in a 4 MiB array built into the library.
    CPU tensors in and out (the output is a CPU tensor: no CUDA tensor is created here either), synchronous.
    Raises Birkhoff4Error for a larger batch.  All calls on one device share that array: do not run two at once
    from different threads.  Make the first call on a device before any stream capture (include/birkhoff4.h).
    `stream`: a torch.cuda.Stream, or None for the current device's legacy default stream (0).
    """
    H_host = _host(H_host, "H_host")
    P_host = torch.empty_like(H_host) if P_host is None else _host(P_host, "P_host", H_host.numel())
    st = ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)
    _check(lib().birkhoff4_forward_host_static(_ptr(H_host), _ptr(P_host), H_host.numel() // 16, tol, max_iter, st))
    return P_host


def birkhoff4_backward_host(P_host, dP_host, dH_host=None):
    P_host = _host(P_host, "P_host")
    dP_host = _host(dP_host, "dP_host", P_host.numel())
    dH_host = torch.empty_like(P_host) if dH_host is None else _host(dH_host, "dH_host", P_host.numel())
    _check(lib().birkhoff4_backward_host(_ptr(P_host), _ptr(dP_host), _ptr(dH_host), P_host.numel() // 16))
    return dH_host


def birkhoff4_forward_backward_host(H_host, dP_host, P_host=None, dH_host=None, tol=1e-6, max_iter=20, want_P=True):
    """host-buffer forward + backward; P stays on the device between the two kernels"""
    H_host = _host(H_host, "H_host")
    dP_host = _host(dP_host, "dP_host", H_host.numel())
    if want_P and P_host is None:
        P_host = torch.empty_like(H_host)
    if P_host is not None:
        _host(P_host, "P_host", H_host.numel())
    dH_host = torch.empty_like(H_host) if dH_host is None else _host(dH_host, "dH_host", H_host.numel())
    _check(lib().birkhoff4_forward_backward_host(_ptr(H_host), _ptr(dP_host), _ptr(P_host), _ptr(dH_host),
                                                 H_host.numel() // 16, tol, max_iter))
    return P_host, dH_host


# ------------------------------------------------------------------------------ include/birkhoff_ot.h
def birkhoff8_forward(H, P=None, tol=2e-6, max_iter=40, iters=None, n_unconverged=None, stream=None):
    """n = 8 Birkhoff projection of exp(H), fp32 CUDA H[B,8,8]"""
    H = _dev(H, torch.float32, "H")
    B = _batch(H, 64, "H")
    P = _out(P, H, "P")
    if iters is not None:
        _dev(iters, torch.int32, "iters", B, H)
    if n_unconverged is not None:
        _dev(n_unconverged, torch.int64, "n_unconverged", 1, H)
    with torch.cuda.device(H.device):
        _check(lib().birkhoff8_forward(_ptr(H), _ptr(P), B, tol, max_iter, _ptr(iters), _ptr(n_unconverged),
                                       _stream(stream, H.device)))
    return P


def birkhoff8_backward(P, dP, dH=None, stream=None):
    """dH = dL/dH from P and dP = dL/dP for the n = 8 projection (fp32 CUDA [B,8,8])"""
    P = _dev(P, torch.float32, "P")
    B = _batch(P, 64, "P")
    dP = _dev(dP, torch.float32, "dP", P.numel(), P)
    dH = _out(dH, P, "dH")
    with torch.cuda.device(P.device):
        _check(lib().birkhoff8_backward(_ptr(P), _ptr(dP), _ptr(dH), B, _stream(stream, P.device)))
    return dH


def entropic_ot_forward(C, a=None, b=None, T=None, eta=1.0, tol=2e-6, max_iter=40, iters=None, n_unconverged=None,
                        stream=None):
    """T = argmin <T,C> - eta h(T) over Pi(a,b) for fp32 CUDA costs C[B,n,m], marginals a[B,n], b[B,m] (or both None)"""
    C = _dev(C, torch.float32, "C")
    if C.dim() != 3:
        raise Birkhoff4Error("C must be [B,n,m]")
    B, n, m = C.shape
    if (a is None) != (b is None):
        raise Birkhoff4Error("give both marginals or neither")
    if a is not None:
        a = _dev(a, torch.float32, "a", B * n, C)
        b = _dev(b, torch.float32, "b", B * m, C)
    T = _out(T, C, "T")
    if iters is not None:
        _dev(iters, torch.int32, "iters", B, C)
    if n_unconverged is not None:
        _dev(n_unconverged, torch.int64, "n_unconverged", 1, C)
    with torch.cuda.device(C.device):
        _check(lib().entropic_ot_forward(_ptr(C), _ptr(a), _ptr(b), _ptr(T), B, n, m, eta, tol, max_iter, _ptr(iters),
                                         _ptr(n_unconverged), _stream(stream, C.device)))
    return T


def entropic_ot_backward(T, G, D=None, eta=1.0, stream=None):
    """D = dl/dC from the forward output T and G = dl/dT (eq. (13)), fp32 CUDA [B,n,m]"""
    T = _dev(T, torch.float32, "T")
    if T.dim() != 3:
        raise Birkhoff4Error("T must be [B,n,m]")
    B, n, m = T.shape
    G = _dev(G, torch.float32, "G", T.numel(), T)
    D = _out(D, T, "D")
    with torch.cuda.device(T.device):
        _check(lib().entropic_ot_backward(_ptr(T), _ptr(G), _ptr(D), B, n, m, eta, _stream(stream, T.device)))
    return D


def birkhoff4_host_release():
    lib().birkhoff4_host_release()


def birkhoff4_version():
    return lib().birkhoff4_version()
