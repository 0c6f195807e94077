"""fp64 CPU oracle for small batched entropic OT (n x m <= 16 x 16) and the n x n Birkhoff projection --
TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/ot_oracle.c for what is computed and the passages it follows).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It shares no code with paper_2606_07574_b200 (the CUDA path) and neither imports the other.

Arrays: M, T, G, D are [B, n, m]; a is [B, n] or None (all ones), b is [B, m] or None; any float dtype is
widened exactly to float64.
"""
import ctypes

import numpy as np

from . import build as _build

_LIB = None
CERTIFY = 1e-12  # a problem whose final Err_ab / sum(a) exceeds this is "oracle-uncertified"


def lib():
    global _LIB
    if _LIB is None:
        L = ctypes.CDLL(_build.build_ot())
        dp, ip = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
        L.oto_forward.argtypes = [dp, dp, dp, dp, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                  ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_double, ip, dp, ctypes.c_int]
        L.oto_forward.restype = ctypes.c_int64
        L.oto_backward.argtypes = [dp, dp, dp, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                   ctypes.c_double, ctypes.c_int]
        L.oto_backward.restype = None
        L.oto_marginal_err.argtypes = [dp, dp, dp, dp, ctypes.c_int64, ctypes.c_int, ctypes.c_int]
        L.oto_marginal_err.restype = None
        L.oto_max_dim.restype = ctypes.c_int
        _LIB = L
    return _LIB


def _c(x, shape=None):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    return a if shape is None else a.reshape(shape)


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _marg(v, B, k):
    return None if v is None else _c(np.broadcast_to(np.asarray(v, np.float64), (B, k)))


def forward(M, a=None, b=None, eta=1.0, tol=1e-14, max_sweeps=200, max_newton=300, nthreads=0, return_info=False):
    """T = argmin <T,M> - eta h(T) over Pi(a,b) (eq. (3)); M is [B,n,m]"""
    M = _c(M)
    B, n, m = M.shape
    a, b = _marg(a, B, n), _marg(b, B, m)
    T = np.empty_like(M)
    tier, err = np.zeros(B, np.int32), np.zeros(B, np.float64)
    bad = lib().oto_forward(_p(M), _p(a), _p(b), _p(T), B, n, m, float(eta), tol, max_sweeps, max_newton, CERTIFY,
                            tier.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _p(err), nthreads)
    if bad < 0:
        raise ValueError("n, m must be in 1..%d" % lib().oto_max_dim())
    if return_info:
        return T, dict(tier=tier, err=err, uncertified=int(bad))
    return T


def backward(T, G, eta=1.0, rcond=1e-13, nthreads=0):
    """D = dl/dM from G = dl/dT (eq. (13)) by the ungauged linearised optimality system"""
    T, G = _c(T), _c(G)
    if T.shape != G.shape:
        raise ValueError("T and G must have the same shape")
    B, n, m = T.shape
    D = np.empty_like(T)
    lib().oto_backward(_p(T), _p(G), _p(D), B, n, m, float(eta), rcond, nthreads)
    return D


def marginal_err(T, a=None, b=None):
    """Err_ab(T) = ||T1 - a||_1 + ||T^T1 - b||_1 per problem (PAPER.md:323 with marginals a, b)"""
    T = _c(T)
    B, n, m = T.shape
    a, b = _marg(a, B, n), _marg(b, B, m)
    e = np.empty(B, np.float64)
    lib().oto_marginal_err(_p(T), _p(a), _p(b), _p(e), B, n, m)
    return e


def birkhoff_forward(H, **kw):
    """P = proj^KL_{B_n}(exp(H)) for [B,n,n] logits: the OT problem with M = -H, eta = 1, a = b = 1"""
    return forward(-_c(H), None, None, 1.0, **kw)


def birkhoff_backward(P, G, **kw):
    """dL/dH = -D for the n x n Birkhoff projection"""
    return -backward(P, G, 1.0, **kw)
